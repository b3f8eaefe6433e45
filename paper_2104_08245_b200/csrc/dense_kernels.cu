// O(n^2) helpers around the batched products (norm bounds, scalings, iterate initialisation,
// iteration control, layout conversion) and the FP32 SIMT product used for FP32-quality steps.
// Every dense buffer is column-major with leading dimension ld (see common.cuh).
#include "common.cuh"

__device__ __forceinline__ int padded_dim(int n) { return (n + NOLSM_TILE_M - 1) / NOLSM_TILE_M * NOLSM_TILE_M; }

__device__ __forceinline__ void atomic_max_nonneg(float *addr, float v) {
  atomicMax(reinterpret_cast<int *>(addr), __float_as_int(v));  // valid for v >= 0
}

// ------------------------------------------------------------------------------------------------
// Upper bound on the spectral radius: rho(A) <= ||A||_2 <= sqrt(||A||_1 ||A||_inf), A = M - mu I
// (rescaling "prior to the sign iteration"; readings 5 and 7).
// norm2[0][m] = ||A||_inf (max abs row sum), norm2[1][m] = ||A||_1 (max abs column sum), from ONE read of
// the matrix.  A block owns a strip of 128 rows; warp w walks the columns c = w, w + 8, ... with one
// 16-byte load per lane (four consecutive rows of the column-major storage).  Row sums accumulate in
// registers and are combined over the eight warps in a fixed order; the strip's share of a column sum
// is a warp reduction written to colpart[m][strip][c], and k_colmax adds the strips in order.  No
// floating-point atomics: the bound is bitwise reproducible.  For a symmetric matrix (S) the column part
// is skipped and ||A||_1 = ||A||_inf.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void load4(const float *p, float (&v)[4]) {
  const float4 q = *reinterpret_cast<const float4 *>(p);
  v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
}
__device__ __forceinline__ void load4(const __half *p, float (&v)[4]) {
  const uint2 q = *reinterpret_cast<const uint2 *>(p);
  const float2 a = __half22float2(*reinterpret_cast<const __half2 *>(&q.x));
  const float2 b = __half22float2(*reinterpret_cast<const __half2 *>(&q.y));
  v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}

template <typename T>
__global__ void __launch_bounds__(256)
k_norm_bound(const int32_t *__restrict__ dims, int ld, int64_t slab, int count, int strips,
             const T *__restrict__ a, float mu, float *__restrict__ norm2, float *__restrict__ colpart) {
  __shared__ float s_row[8][128];
  const int mat = blockIdx.y;
  const int n = dims[mat];
  const int base = blockIdx.x * 128;
  if (base >= n) return;
  const T *aj = a + (int64_t)mat * slab;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = base + 4 * lane;
  float racc[4] = {0.f, 0.f, 0.f, 0.f};
  float *cp = colpart ? colpart + ((int64_t)mat * strips + blockIdx.x) * ld : nullptr;
  for (int c = warp; c < n; c += 8) {
    float v[4];
    load4(aj + (int64_t)c * ld + r0, v);
    float cs = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int r = r0 + i;
      float x = r < n ? v[i] : 0.f;     // rows beyond n may hold stale data
      if (r == c) x -= mu;
      x = fabsf(x);
      racc[i] += x;
      cs += x;
    }
    if (cp) {
      for (int d = 16; d > 0; d >>= 1) cs += __shfl_xor_sync(0xffffffffu, cs, d);
      if (lane == 0) cp[c] = cs;
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) s_row[warp][4 * lane + i] = racc[i];
  __syncthreads();
  if (threadIdx.x < 128) {
    float rs = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) rs += s_row[w][threadIdx.x];
    for (int d = 16; d > 0; d >>= 1) rs = fmaxf(rs, __shfl_xor_sync(0xffffffffu, rs, d));
    if (lane == 0) {
      atomic_max_nonneg(&norm2[mat], rs);
      if (!cp) atomic_max_nonneg(&norm2[count + mat], rs);
    }
  }
}

__global__ void __launch_bounds__(256)
k_colmax(const int32_t *__restrict__ dims, int ld, int count, int strips, const float *__restrict__ colpart,
         float *__restrict__ norm2) {
  __shared__ float s_max[8];
  const int mat = blockIdx.x;
  const int n = dims[mat];
  const int ns = (n + 127) / 128;
  const float *cp = colpart + (int64_t)mat * strips * ld;
  float m = 0.f;
  for (int c = threadIdx.x; c < n; c += blockDim.x) {
    float cs = 0.f;
    for (int s = 0; s < ns; ++s) cs += cp[(int64_t)s * ld + c];
    m = fmaxf(m, cs);
  }
  for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
  if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) m = fmaxf(m, s_max[w]);
    norm2[count + mat] = m;
  }
}

template <typename T>
static cudaError_t norm_bound_impl(const nolsm_batch *b, const T *a, float mu, bool symmetric, float *norm2,
                                   cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  cudaError_t e = cudaMemsetAsync(norm2, 0, sizeof(float) * 2 * b->count, st);
  if (e != cudaSuccess) return e;
  const int strips = (b->ld + 127) / 128;
  dim3 grid((b->max_n + 127) / 128, b->count);
  k_norm_bound<T><<<grid, 256, 0, st>>>(b->d_dims, b->ld, (int64_t)b->ld * b->ld, b->count, strips, a, mu, norm2,
                                        symmetric ? nullptr : b->d_colpart);
  if (!symmetric) k_colmax<<<b->count, 256, 0, st>>>(b->d_dims, b->ld, b->count, strips, b->d_colpart, norm2);
  return cudaGetLastError();
}
cudaError_t launch_norm_bound(const nolsm_batch *b, const float *a, float mu, bool symmetric, float *norm2,
                              cudaStream_t st) {
  return norm_bound_impl(b, a, mu, symmetric, norm2, st);
}
// the same bound from an FP16 matrix
cudaError_t launch_norm_bound16(const nolsm_batch *b, const __half *a, float mu, float *norm2, cudaStream_t st) {
  return norm_bound_impl(b, a, mu, false, norm2, st);
}

// s_j of X0 = (B - mu I)/s_j (reading 5) from the norm bound, inflated by `slack` where the bound was taken on an
// approximation of the matrix
__global__ void k_x0_scale(int count, const float *__restrict__ norm2, float factor, float slack,
                           float *__restrict__ scale_out) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m < count) scale_out[m] = fmaxf(slack * factor * sqrtf(norm2[m] * norm2[count + m]), 1e-30f);
}
cudaError_t launch_x0_scale(const nolsm_batch *b, const float *norm2, float slack, float *scale_out, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_x0_scale<<<(b->count + 255) / 256, 256, 0, st>>>(b->count, norm2, b->sign_scale, slack, scale_out);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Element-wise passes over the padded P x P part of every submatrix.  One thread = four consecutive
// rows of one column (16-byte FP32 accesses, 8-byte FP16 stores; ld is a multiple of 128, so every
// access is aligned); blockIdx.y = submatrix.
// ------------------------------------------------------------------------------------------------
struct Elem4 { int r, c, n; int64_t off; };

__device__ __forceinline__ bool elem4(const int32_t *__restrict__ dims, int ld, int64_t slab, Elem4 &e) {
  const int mat = blockIdx.y;
  e.n = dims[mat];
  const int P = padded_dim(e.n);
  const int q = P >> 2;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= q * P) return false;
  e.c = i / q;
  e.r = (i - e.c * q) << 2;
  e.off = (int64_t)mat * slab + (int64_t)e.c * ld + e.r;
  return true;
}

__device__ __forceinline__ void store_half4(__half *dst, const float (&v)[4]) {
  const __half2 a = __floats2half2_rn(v[0], v[1]), b = __floats2half2_rn(v[2], v[3]);
  uint2 pk;
  pk.x = *reinterpret_cast<const uint32_t *>(&a);
  pk.y = *reinterpret_cast<const uint32_t *>(&b);
  *reinterpret_cast<uint2 *>(dst) = pk;
}

// hi = fp16(v), lo = fp16((v - hi) * 2^11): the split operands of the FP32-quality products
__device__ __forceinline__ void store_split4(__half *hi, __half *lo, const float (&v)[4]) {
  if (lo == nullptr) {   // plain FP16 copy: none of the lo arithmetic (these passes are issue-bound, not HBM-bound)
    store_half4(hi, v);
    return;
  }
  float h[4], l[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    h[i] = __half2float(__float2half_rn(v[i]));
    l[i] = (v[i] - h[i]) * 2048.f;
  }
  store_half4(hi, h);
  store_half4(lo, l);
}

static dim3 elem4_grid(const nolsm_batch *b) {
  const int P = round_up(b->max_n, NOLSM_TILE_M);
  return dim3((unsigned)(((int64_t)(P >> 2) * P + 255) / 256), (unsigned)b->count);
}

// Eq. 15: Y0 = T_j(S)/s_S, Z0 = I with s_S = 1/2 max(1, sqrt(||S||_1 ||S||_inf)) >=
// lambda_max(S)/2 (reading 7): the spectrum of Y0 lies in (0, 2], inside the interval (0, 3) on
// which v -> v (3 - v)^2 / 4 converges to 1, and roughly centred on 1, which saves one iteration over
// scaling to (0, 1].  The padded part of S is the identity, so Y0 there is 1/s_S <= 2.
// X0 = A/s with s = sqrt(||A||_1 ||A||_inf)/1.5 >= rho(A)/1.5 (reading 5): every eigenvalue of X0 lies in
// [-1.5, 1.5], inside the interval |x| < sqrt(3) on which Eq. 9 converges to sign(x).
// Both factors come from the batch (1 under NOLSM_FLAG_UNIT_SCALE).
__global__ void __launch_bounds__(256)
k_init_inverse(const int32_t *__restrict__ dims, int ld, int64_t slab, int count,
               const float *__restrict__ s, const float *__restrict__ norm2, float *__restrict__ y32,
               float *__restrict__ z32, __half *__restrict__ y16, __half *__restrict__ z16,
               __half *__restrict__ y16_lo, __half *__restrict__ z16_lo, float *__restrict__ scale_out,
               float factor) {
  Elem4 e;
  if (!elem4(dims, ld, slab, e)) return;
  const int mat = blockIdx.y;
  const float sc = factor * fmaxf(1.f, sqrtf(norm2[mat] * norm2[count + mat]));  // max(1, .) covers the unit padding
  if (e.r == 0 && e.c == 0) scale_out[mat] = sc;
  const float4 sv = *reinterpret_cast<const float4 *>(s + e.off);
  const float inv = 1.f / sc;
  const float y[4] = {sv.x * inv, sv.y * inv, sv.z * inv, sv.w * inv};
  float z[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) z[i] = (e.r + i == e.c) ? 1.f : 0.f;
  if (y32) {
    *reinterpret_cast<float4 *>(y32 + e.off) = make_float4(y[0], y[1], y[2], y[3]);
    *reinterpret_cast<float4 *>(z32 + e.off) = make_float4(z[0], z[1], z[2], z[3]);
  }
  if (y16) {
    store_split4(y16 + e.off, y16_lo ? y16_lo + e.off : nullptr, y);
    store_split4(z16 + e.off, z16_lo ? z16_lo + e.off : nullptr, z);
  }
}

cudaError_t launch_init_inverse(const nolsm_batch *b, const float *s, const float *norm2, float *y32,
                                float *z32, __half *y16, __half *z16, __half *y16_lo, __half *z16_lo,
                                float *scale_out, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_init_inverse<<<elem4_grid(b), 256, 0, st>>>(b->d_dims, b->ld, (int64_t)b->ld * b->ld, b->count, s, norm2,
                                                y32, z32, y16, z16, y16_lo, z16_lo, scale_out, b->inv_scale);
  return cudaGetLastError();
}

// Eq. 15-16 with the first iteration done in closed form: Z0 = I gives E0 = I - Z0 Y0 = I - Y0 and
// Z1 = Z0 + 1/2 E0 Z0 = 3/2 I - 1/2 Y0 without any product; only Y1 = Y0 + 1/2 Y0 E0 needs one.
// Writes Y0 (FP32 master + FP16 operand), E0 (FP16 operand) and Z1 (FP32 master + FP16 operand).
__global__ void __launch_bounds__(256)
k_init_inverse_first(const int32_t *__restrict__ dims, int ld, int64_t slab, int count,
                     const float *__restrict__ s, const float *__restrict__ norm2, float *__restrict__ y32,
                     float *__restrict__ z32, __half *__restrict__ y16, __half *__restrict__ y16_lo,
                     __half *__restrict__ z16, __half *__restrict__ z16_lo, __half *__restrict__ e16,
                     __half *__restrict__ e16_lo, float *__restrict__ scale_out, float factor) {
  Elem4 e;
  if (!elem4(dims, ld, slab, e)) return;
  const int mat = blockIdx.y;
  const float sc = factor * fmaxf(1.f, sqrtf(norm2[mat] * norm2[count + mat]));
  if (e.r == 0 && e.c == 0) scale_out[mat] = sc;
  const float4 sv = *reinterpret_cast<const float4 *>(s + e.off);
  const float inv = 1.f / sc;   // one reciprocal instead of four IEEE divisions: the pass is issue-bound
  const float y[4] = {sv.x * inv, sv.y * inv, sv.z * inv, sv.w * inv};
  float ev[4], z[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float d = (e.r + i == e.c) ? 1.f : 0.f;
    ev[i] = d - y[i];
    z[i] = fmaf(0.5f, ev[i], d);
  }
  if (y32) {   // FP32 masters (not kept when the iterates live in FP16 only)
    *reinterpret_cast<float4 *>(y32 + e.off) = make_float4(y[0], y[1], y[2], y[3]);
    *reinterpret_cast<float4 *>(z32 + e.off) = make_float4(z[0], z[1], z[2], z[3]);
  }
  store_split4(y16 + e.off, y16_lo ? y16_lo + e.off : nullptr, y);
  store_split4(z16 + e.off, z16_lo ? z16_lo + e.off : nullptr, z);
  store_split4(e16 + e.off, e16_lo ? e16_lo + e.off : nullptr, ev);
}

cudaError_t launch_init_inverse_first(const nolsm_batch *b, const float *s, const float *norm2, float *y32,
                                      float *z32, __half *y16, __half *y16_lo, __half *z16, __half *z16_lo,
                                      __half *e16, __half *e16_lo, float *scale_out, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_init_inverse_first<<<elem4_grid(b), 256, 0, st>>>(b->d_dims, b->ld, (int64_t)b->ld * b->ld, b->count, s, norm2,
                                                      y32, z32, y16, y16_lo, z16, z16_lo, e16, e16_lo, scale_out,
                                                      b->inv_scale);
  return cudaGetLastError();
}

// Lean start of Eq. 15-17 when the iterates live in FP16 only (FP16 mode with a refinement behind the iteration):
// Y0 = S/s_S is never written -- with Z0 = I the first iteration gives Z1 = 3/2 I - 1/2 Y0 element-wise and
// Y1 = Y0 + 1/2 Y0 (I - Y0) = Y0 Z1 = (S_hi Z1)/s_S as ONE product whose left operand is the FP16 copy of S the
// builder wrote (scaled by 1/s_S in the product's epilogue, so Y0 = S_hi/s_S carries no second rounding).
// Reads the split S (4 bytes per element), writes Z1 (2 bytes) instead of reading 4 and writing 6.
// Element-wise passes, eight rows per thread: thread t of a block owns rows 8t..8t+7 (one 16-byte FP16 access, two
// for FP32) of kElemCols consecutive columns -- no index division, 16-byte accesses, all loads of a thread issued
// before the first use (the four-element version was bound by instruction issue, not by HBM).
constexpr int kElemCols = 4;
static dim3 elem8_grid(const nolsm_batch *b) {
  const int P = round_up(b->max_n, NOLSM_TILE_M);
  return dim3((unsigned)((P + kElemCols - 1) / kElemCols), (unsigned)b->count);
}
static int elem8_threads(const nolsm_batch *b) { return std::min(256, (round_up(b->max_n, NOLSM_TILE_M) / 8 + 31) / 32 * 32); }

__device__ __forceinline__ void unpack8(const uint4 &q, float (&v)[8]) {
  const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&w[i]));
    v[2 * i] = f.x; v[2 * i + 1] = f.y;
  }
}
__device__ __forceinline__ uint4 pack8(const float (&v)[8]) {
  uint32_t w[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const __half2 h = __floats2half2_rn(v[2 * i], v[2 * i + 1]);
    w[i] = *reinterpret_cast<const uint32_t *>(&h);
  }
  return make_uint4(w[0], w[1], w[2], w[3]);
}
// hi = fp16(v), lo = fp16((v - hi) * 2^11)
__device__ __forceinline__ void split8(const float (&v)[8], uint4 &hi, uint4 &lo) {
  hi = pack8(v);
  float h[8], l[8];
  unpack8(hi, h);
#pragma unroll
  for (int i = 0; i < 8; ++i) l[i] = (v[i] - h[i]) * 2048.f;
  lo = pack8(l);
}

__global__ void __launch_bounds__(256)
k_init_z1(const int32_t *__restrict__ dims, int ld, int64_t slab, int count, const __half *__restrict__ s_hi,
          const __half *__restrict__ s_lo, const float *__restrict__ norm2, __half *__restrict__ z16,
          float *__restrict__ scale_out, float factor) {
  const int mat = blockIdx.y;
  const int P = padded_dim(dims[mat]);
  const int c0 = blockIdx.x * kElemCols;
  if (c0 >= P) return;
  const float sc = factor * fmaxf(1.f, sqrtf(norm2[mat] * norm2[count + mat]));
  if (threadIdx.x == 0 && c0 == 0) scale_out[mat] = sc;
  for (int r = 8 * threadIdx.x; r < P; r += 8 * blockDim.x) {
  const int64_t off = (int64_t)mat * slab + (int64_t)c0 * ld + r;
  uint4 hq[kElemCols], lq[kElemCols];
#pragma unroll
  for (int u = 0; u < kElemCols; ++u) {   // P is a multiple of 128: a block's columns are all inside or all outside
    hq[u] = *reinterpret_cast<const uint4 *>(s_hi + off + (int64_t)u * ld);
    lq[u] = *reinterpret_cast<const uint4 *>(s_lo + off + (int64_t)u * ld);
  }
  const float inv = -0.5f / sc;
#pragma unroll
  for (int u = 0; u < kElemCols; ++u) {
    float h[8], l[8], z[8];
    unpack8(hq[u], h);
    unpack8(lq[u], l);
#pragma unroll
    for (int i = 0; i < 8; ++i) z[i] = fmaf(fmaf(l[i], 1.f / 2048.f, h[i]), inv, (r + i == c0 + u) ? 1.5f : 0.f);
    *reinterpret_cast<uint4 *>(z16 + off + (int64_t)u * ld) = pack8(z);
  }
  }
}

cudaError_t launch_init_z1(const nolsm_batch *b, const __half *s_hi, const __half *s_lo, const float *norm2, __half *z16,
                           float *scale_out, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_init_z1<<<elem8_grid(b), elem8_threads(b), 0, st>>>(b->d_dims, b->ld, (int64_t)b->ld * b->ld, b->count, s_hi, s_lo,
                                                         norm2, z16, scale_out, b->inv_scale);
  return cudaGetLastError();
}

// The final iterate of a ping-pong chain lives in one of two split pairs, by the parity of the submatrix's iteration
// count ((iters[m] + 1) & 1, ChainProgram::parity_from_iters).  This copies pair 0 onto pair 1 where the parity is 0,
// so that afterwards every submatrix has it in pair 1 (for consumers that run after iters has been reused).
__global__ void __launch_bounds__(256)
k_canon_pair(const int32_t *__restrict__ dims, const int32_t *__restrict__ iters, int ld, int64_t slab,
             const __half *__restrict__ hi0, const __half *__restrict__ lo0, __half *__restrict__ hi1,
             __half *__restrict__ lo1) {
  const int mat = blockIdx.y;
  if (((iters[mat] + 1) & 1) != 0) return;
  const int P = padded_dim(dims[mat]);
  const int c0 = blockIdx.x * kElemCols;
  if (c0 >= P) return;
  for (int r = 8 * threadIdx.x; r < P; r += 8 * blockDim.x) {
    const int64_t off = (int64_t)mat * slab + (int64_t)c0 * ld + r;
    uint4 h[kElemCols], l[kElemCols];
#pragma unroll
    for (int u = 0; u < kElemCols; ++u) {
      h[u] = *reinterpret_cast<const uint4 *>(hi0 + off + (int64_t)u * ld);
      l[u] = *reinterpret_cast<const uint4 *>(lo0 + off + (int64_t)u * ld);
    }
#pragma unroll
    for (int u = 0; u < kElemCols; ++u) {
      *reinterpret_cast<uint4 *>(hi1 + off + (int64_t)u * ld) = h[u];
      *reinterpret_cast<uint4 *>(lo1 + off + (int64_t)u * ld) = l[u];
    }
  }
}

cudaError_t launch_canon_pair(const nolsm_batch *b, const int32_t *iters, const __half *hi0, const __half *lo0,
                              __half *hi1, __half *lo1, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_canon_pair<<<elem8_grid(b), elem8_threads(b), 0, st>>>(b->d_dims, iters, b->ld, (int64_t)b->ld * b->ld, hi0, lo0,
                                                            hi1, lo1);
  return cudaGetLastError();
}

// X0 = (B - mu I)/s  (Eq. 9 with the rescaling of PAPER.md:138), s from the norm bound or from the
// caller (scale_in, dense microbench).  Padded diagonal = 1: a fixed point of the iteration that adds
// nothing to the residual (reading 19).
__global__ void __launch_bounds__(256)
k_make_x0(const int32_t *__restrict__ dims, int ld, int64_t slab, int count,
          const float *__restrict__ bmat, float mu, const float *__restrict__ norm2,
          const float *__restrict__ scale_in, float *__restrict__ x32, __half *__restrict__ x16,
          __half *__restrict__ x16_lo, float *__restrict__ scale_out, float factor) {
  Elem4 e;
  if (!elem4(dims, ld, slab, e)) return;
  const int mat = blockIdx.y;
  float sc = scale_in ? scale_in[mat] : factor * sqrtf(norm2[mat] * norm2[count + mat]);
  sc = fmaxf(sc, 1e-30f);
  const float inv = 1.f / sc;
  if (e.r == 0 && e.c == 0 && scale_out) scale_out[mat] = sc;
  const float4 bv = *reinterpret_cast<const float4 *>(bmat + e.off);
  const float in[4] = {bv.x, bv.y, bv.z, bv.w};
  float v[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = e.r + i;
    if (r < e.n && e.c < e.n) v[i] = (in[i] - (r == e.c ? mu : 0.f)) * inv;
    else v[i] = (r == e.c) ? 1.f : 0.f;
  }
  if (x32) *reinterpret_cast<float4 *>(x32 + e.off) = make_float4(v[0], v[1], v[2], v[3]);
  if (x16) store_split4(x16 + e.off, x16_lo ? x16_lo + e.off : nullptr, v);
}

// the same for the split iterate of the tensor-core engine (no FP32 copy), eight rows per thread
__global__ void __launch_bounds__(256)
k_make_x0_split(const int32_t *__restrict__ dims, int ld, int64_t slab, int count, const float *__restrict__ bmat,
                float mu, const float *__restrict__ norm2, const float *__restrict__ scale_in,
                __half *__restrict__ x16, __half *__restrict__ x16_lo, float *__restrict__ scale_out, float factor) {
  const int mat = blockIdx.y;
  const int n = dims[mat];
  const int P = padded_dim(n);
  const int c0 = blockIdx.x * kElemCols;
  if (c0 >= P) return;
  float sc = scale_in ? scale_in[mat] : factor * sqrtf(norm2[mat] * norm2[count + mat]);
  sc = fmaxf(sc, 1e-30f);
  const float inv = 1.f / sc;
  if (threadIdx.x == 0 && c0 == 0 && scale_out) scale_out[mat] = sc;
  for (int r = 8 * threadIdx.x; r < P; r += 8 * blockDim.x) {
  const int64_t off = (int64_t)mat * slab + (int64_t)c0 * ld + r;
  float4 bq[kElemCols][2];
#pragma unroll
  for (int u = 0; u < kElemCols; ++u) {
    const float4 *src = reinterpret_cast<const float4 *>(bmat + off + (int64_t)u * ld);
    bq[u][0] = src[0];
    bq[u][1] = src[1];
  }
#pragma unroll
  for (int u = 0; u < kElemCols; ++u) {
    const int c = c0 + u;
    const float in[8] = {bq[u][0].x, bq[u][0].y, bq[u][0].z, bq[u][0].w, bq[u][1].x, bq[u][1].y, bq[u][1].z, bq[u][1].w};
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if (r + i < n && c < n) v[i] = (in[i] - (r + i == c ? mu : 0.f)) * inv;
      else v[i] = (r + i == c) ? 1.f : 0.f;
    }
    uint4 hi, lo;
    split8(v, hi, lo);
    *reinterpret_cast<uint4 *>(x16 + off + (int64_t)u * ld) = hi;
    *reinterpret_cast<uint4 *>(x16_lo + off + (int64_t)u * ld) = lo;
  }
  }
}

cudaError_t launch_make_x0(const nolsm_batch *b, const float *bmat, float mu, const float *norm2,
                           const float *scale_in, float *x32, __half *x16, __half *x16_lo, float *scale_out,
                           cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  if (!x32 && x16 && x16_lo) {
    k_make_x0_split<<<elem8_grid(b), elem8_threads(b), 0, st>>>(b->d_dims, b->ld, (int64_t)b->ld * b->ld, b->count, bmat,
                                                                 mu, norm2, scale_in, x16, x16_lo, scale_out,
                                                                 b->sign_scale);
    return cudaGetLastError();
  }
  k_make_x0<<<elem4_grid(b), 256, 0, st>>>(b->d_dims, b->ld, (int64_t)b->ld * b->ld, b->count, bmat, mu, norm2,
                                           scale_in, x32, x16, x16_lo, scale_out, b->sign_scale);
  return cudaGetLastError();
}

// Scaled Newton-Schulz start (Chen & Chow's scaling of Eq. 9): with a lower bound l
// on the moduli of the eigenvalues of X (all <= 1), X <- 1/2 a X (3I - a^2 X^2) with a = sqrt(3 / (1 + l + l^2))
// maps [l, 1] onto [l', 1] with l' = 1/2 a l (3 - a^2 l^2) = the image of both ends: the largest l' any a gives.
// Any a in [1, sqrt 3] keeps a |x| <= sqrt 3, so a wrong bound costs iterations, never convergence.
// X0 has |x| <= 1.5, so iteration 0 is the plain one (a = 1), which brings the spectrum into [-1, 1].
__global__ void k_alpha_schedule(int count, const float *__restrict__ scale, float gap, float *__restrict__ tab) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= count) return;
  float l = fminf(gap / scale[m], 1.f);
  tab[m * 8] = 1.f;
  l = 0.5f * l * (3.f - l * l);
  for (int k = 1; k < 8; ++k) {
    float a = sqrtf(3.f / (1.f + l + l * l));
    if (a < 1.02f) a = 1.f;
    tab[m * 8 + k] = a;
    l = 0.5f * a * l * (3.f - a * a * l * l);
  }
}

cudaError_t launch_alpha_schedule(const nolsm_batch *b, const float *scale, float gap, float *alpha_tab,
                                  cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_alpha_schedule<<<(b->count + 127) / 128, 128, 0, st>>>(b->count, scale, gap, alpha_tab);
  return cudaGetLastError();
}

// dst = src * f (f = scale[m], 1/scale[m] or 1), FP32 and/or FP16 (hi [+ lo*2^11]) copies over the
// padded extent.  Hands FP32 results to the tensor-core path.
__global__ void __launch_bounds__(256)
k_scale_copy(const int32_t *__restrict__ dims, int ld, int64_t slab, const float *__restrict__ src,
             const float *__restrict__ scale, int invert, float *__restrict__ dst32,
             __half *__restrict__ dst16, __half *__restrict__ dst16_lo) {
  Elem4 e;
  if (!elem4(dims, ld, slab, e)) return;
  float f = 1.f;
  if (scale) f = invert ? 1.f / scale[blockIdx.y] : scale[blockIdx.y];
  const float4 sv = *reinterpret_cast<const float4 *>(src + e.off);
  const float v[4] = {sv.x * f, sv.y * f, sv.z * f, sv.w * f};
  if (dst32) *reinterpret_cast<float4 *>(dst32 + e.off) = make_float4(v[0], v[1], v[2], v[3]);
  if (dst16) store_split4(dst16 + e.off, dst16_lo ? dst16_lo + e.off : nullptr, v);
}

cudaError_t launch_scale_copy(const nolsm_batch *b, const float *src, const float *scale, int invert,
                              float *dst32, __half *dst16, __half *dst16_lo, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_scale_copy<<<elem4_grid(b), 256, 0, st>>>(b->d_dims, b->ld, (int64_t)b->ld * b->ld, src, scale, invert,
                                              dst32, dst16, dst16_lo);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Iteration control (stop rule, reading 9).  state[m] holds the LAST iteration index the
// submatrix executes (INT_MAX while undecided); a product of iteration k runs for m iff k <= state[m].
// After the first product of iteration k (which produced the residual) this kernel decides:
// r_k < tol (or the fixed count / the cap reached) -> iteration k is finished and is the last one.
// lockstep: everybody stops together once the slowest has met the test (FP32 ping-pong buffers).
// phase 0 = reset for a new iteration sequence.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_control(int count, const int32_t *__restrict__ dims, int32_t *__restrict__ state,
          int32_t *__restrict__ iters, const float *__restrict__ resid2, float *__restrict__ lastres,
          int32_t *__restrict__ active, int phase, int iter, float tol, int max_iter, int fixed_iter,
          int lockstep) {
  __shared__ int s_cnt;
  if (threadIdx.x == 0) s_cnt = 0;
  __syncthreads();
  if (phase == 0) {
    for (int m = threadIdx.x; m < count; m += blockDim.x) {
      state[m] = 0x7fffffff;
      iters[m] = 0;
      lastres[m] = -1.f;
    }
    return;
  }
  int mine = 0;
  for (int m = threadIdx.x; m < count; m += blockDim.x) {
    if (iter <= state[m]) {
      const float r = sqrtf(fmaxf(resid2[m], 0.f) / (float)dims[m]);
      lastres[m] = r;
      iters[m] = iter + 1;
      bool stop;
      if (fixed_iter > 0) stop = (iter + 1 >= fixed_iter);
      else stop = (r < tol) || !(r == r);
      if (iter + 1 >= max_iter) stop = true;
      if (!stop) mine++;
      else if (!lockstep) state[m] = iter;
    }
  }
  atomicAdd(&s_cnt, mine);
  __syncthreads();
  const int total = s_cnt;
  if (lockstep && total == 0) {
    for (int m = threadIdx.x; m < count; m += blockDim.x)
      if (iter <= state[m]) state[m] = iter;
  }
  if (threadIdx.x == 0) active[iter] = total;
}

cudaError_t launch_control(const nolsm_batch *b, int phase, int iter, float tol, int max_iter,
                           int fixed_iter, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  const int lockstep = phase >> 4;
  k_control<<<1, 256, 0, st>>>(b->count, b->d_dims, b->d_state, b->d_iters,
                               b->d_resid2 + (size_t)(iter % NOLSM_MAX_RESID_SLOTS) * b->count,
                               b->d_lastres, b->d_active, phase & 15, iter, tol, max_iter, fixed_iter,
                               lockstep);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Layout conversion between the caller's row-major n x n matrices and the padded column-major slabs
// (dense microbench entry, test entry, nolsm_batch_read).  32x32 shared-memory transpose.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_pack(const float *__restrict__ src, int n, int ld, int64_t slab, float *__restrict__ dst, int P,
       int pad_identity) {
  __shared__ float t[32][33];
  const int mat = blockIdx.z;
  const float *s = src + (int64_t)mat * n * n;
  float *d = dst + (int64_t)mat * slab;
  const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int i = ty; i < 32; i += 8) {
    const int r = r0 + i, c = c0 + tx;
    float v = 0.f;
    if (r < n && c < n) v = s[(int64_t)r * n + c];
    else if (pad_identity && r == c) v = 1.f;
    t[i][tx] = v;
  }
  __syncthreads();
  for (int i = ty; i < 32; i += 8) {
    const int c = c0 + i, r = r0 + tx;
    if (r < P && c < P) d[(int64_t)c * ld + r] = t[tx][i];
  }
}

cudaError_t launch_pack(const float *src_rowmajor, int n, int batch, int ld, float *dst, int pad_identity,
                        cudaStream_t st) {
  if (batch == 0) return cudaSuccess;
  const int P = round_up(n, NOLSM_TILE_M);
  dim3 grid((P + 31) / 32, (P + 31) / 32, batch);
  k_pack<<<grid, 256, 0, st>>>(src_rowmajor, n, ld, (int64_t)ld * ld, dst, P, pad_identity);
  return cudaGetLastError();
}

__global__ void __launch_bounds__(256)
k_unpack(const float *__restrict__ src, const float *__restrict__ src_alt,
         const int32_t *__restrict__ parity, int ld, int64_t slab, int n, float *__restrict__ dst) {
  __shared__ float t[32][33];
  const int mat = blockIdx.z;
  const float *s = ((src_alt && parity && (parity[mat] & 1)) ? src_alt : src) + (int64_t)mat * slab;
  float *d = dst + (int64_t)mat * n * n;
  const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int i = ty; i < 32; i += 8) {
    const int c = c0 + i, r = r0 + tx;
    t[i][tx] = (r < n && c < n) ? s[(int64_t)c * ld + r] : 0.f;
  }
  __syncthreads();
  for (int i = ty; i < 32; i += 8) {
    const int r = r0 + i, c = c0 + tx;
    if (r < n && c < n) d[(int64_t)r * n + c] = t[tx][i];
  }
}

cudaError_t launch_unpack(const float *src, int ld, int64_t slab, const int32_t *iters_parity,
                          const float *src_alt, int n, int batch, float *dst_rowmajor, cudaStream_t st) {
  if (batch == 0) return cudaSuccess;
  dim3 grid((n + 31) / 32, (n + 31) / 32, batch);
  k_unpack<<<grid, 256, 0, st>>>(src, src_alt, iters_parity, ld, slab, n, dst_rowmajor);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// FP32 SIMT batched product with the engine's epilogues: 128x128 tile, 256 threads, 8x8 per thread,
// K step 16.  Bound by the plain FP32 pipes; used for the FP32-quality steps until the split-FP16
// tensor path takes over, and as the numerical reference of the tcgen05 kernels in the tests.
// ------------------------------------------------------------------------------------------------
#define SG_BK 16

__global__ void __launch_bounds__(256)
k_gemm_simt(GemmParams p) {
  __shared__ float As[SG_BK][128];
  __shared__ float Bs[SG_BK][132];
  for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
    const TileDesc td = p.tiles[t];
    if (p.state && p.iter > p.state[td.mat]) continue;
    const int n = p.dims[td.mat];
    const int K = (n + SG_BK - 1) / SG_BK * SG_BK;  // padded region is valid (identity / zero)
    const float *A = p.a32 + (int64_t)td.mat * p.slab;
    const float *B = p.b32 + (int64_t)td.mat * p.slab;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    float acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;
    for (int k0 = 0; k0 < K; k0 += SG_BK) {
      __syncthreads();
      // A tile: columns k0..k0+15, rows m0..m0+127 (contiguous along rows)
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int idx = threadIdx.x + i * 256;      // 512 float4
        const int kk = idx >> 5, r4 = (idx & 31) * 4;
        const float4 v = *reinterpret_cast<const float4 *>(A + (int64_t)(k0 + kk) * p.ld + td.m0 + r4);
        *reinterpret_cast<float4 *>(&As[kk][r4]) = v;
      }
      // B tile: columns n0..n0+127 of B, rows k0..k0+15 (contiguous along k) -> Bs[k][n]
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int idx = threadIdx.x + i * 256;
        const int nn = idx >> 2, k4 = (idx & 3) * 4;
        const float4 v = *reinterpret_cast<const float4 *>(B + (int64_t)(td.n0 + nn) * p.ld + k0 + k4);
        Bs[k4 + 0][nn] = v.x; Bs[k4 + 1][nn] = v.y; Bs[k4 + 2][nn] = v.z; Bs[k4 + 3][nn] = v.w;
      }
      __syncthreads();
#pragma unroll
      for (int kk = 0; kk < SG_BK; ++kk) {
        float a[8], b[8];
        *reinterpret_cast<float4 *>(&a[0]) = *reinterpret_cast<const float4 *>(&As[kk][tx * 4]);
        *reinterpret_cast<float4 *>(&a[4]) = *reinterpret_cast<const float4 *>(&As[kk][64 + tx * 4]);
        *reinterpret_cast<float4 *>(&b[0]) = *reinterpret_cast<const float4 *>(&Bs[kk][ty * 4]);
        *reinterpret_cast<float4 *>(&b[4]) = *reinterpret_cast<const float4 *>(&Bs[kk][64 + ty * 4]);
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
          for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
      }
    }
    // epilogue: thread owns rows {tx*4..+3, 64+tx*4..+3} x cols {ty*4..+3, 64+ty*4..+3}
    float ss = 0.f;
    const int64_t base = (int64_t)td.mat * p.slab;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int c = td.n0 + (j < 4 ? ty * 4 + j : 64 + ty * 4 + (j - 4));
#pragma unroll
      for (int ih = 0; ih < 2; ++ih) {
        const int r = td.m0 + (ih ? 64 + tx * 4 : tx * 4);
        const int64_t off = base + (int64_t)c * p.ld + r;
        float4 o;
        float *ov = reinterpret_cast<float *>(&o);
        if (p.mode == EPI_IDENT) {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float v = ((r + i == c) ? 1.f : 0.f) - acc[ih * 4 + i][j];
            ov[i] = v;
            if (r + i < n && c < n) ss = fmaf(v, v, ss);
          }
        } else {
          float4 ci = make_float4(0.f, 0.f, 0.f, 0.f);
          if (p.beta != 0.f) ci = *reinterpret_cast<const float4 *>(p.cin32 + off);
          const float *cv = reinterpret_cast<const float *>(&ci);
          const float al = p.alpha_div ? p.alpha / p.alpha_div[td.mat] : p.alpha;
#pragma unroll
          for (int i = 0; i < 4; ++i) ov[i] = fmaf(al, acc[ih * 4 + i][j], p.beta * cv[i]);
        }
        if (p.cout32) *reinterpret_cast<float4 *>(p.cout32 + off) = o;
        if (p.cout16) {
          __half2 h01 = __floats2half2_rn(ov[0], ov[1]), h23 = __floats2half2_rn(ov[2], ov[3]);
          uint2 pk;
          pk.x = *reinterpret_cast<uint32_t *>(&h01);
          pk.y = *reinterpret_cast<uint32_t *>(&h23);
          *reinterpret_cast<uint2 *>(p.cout16 + off) = pk;
        }
      }
    }
    if (p.mode == EPI_IDENT && p.resid2) {
      for (int d = 16; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
      if ((threadIdx.x & 31) == 0) atomicAdd(&p.resid2[td.mat], ss);
    }
  }
}

cudaError_t launch_gemm_simt(const GemmParams &p, cudaStream_t st) {
  if (p.n_tiles == 0) return cudaSuccess;
  int grid = p.n_tiles < 148 * 8 ? p.n_tiles : 148 * 8;
  k_gemm_simt<<<grid, 256, 0, st>>>(p);
  return cudaGetLastError();
}
