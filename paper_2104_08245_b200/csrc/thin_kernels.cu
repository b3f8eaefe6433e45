// Thin products of the hot path: C = A V with A a dense n x n submatrix held as FP16 planes (hi [+ lo * 2^-11], the
// split form of DESIGN.md reading 12) and V its n x 6 "own" operand.  They are bound by reading A once from HBM
// (DESIGN.md 5.2); on the FP32 pipe the 6 FMAs per element plus conversions exhaust the issue slots at about half of
// the HBM rate, so the contraction itself runs on mma.sync (m16n8k16, FP16 operands, FP32 accumulate) -- a thin GEMM
// where the tensor core only takes the arithmetic out of the way of the loads; tcgen05/TMEM would add nothing at 6
// columns.
//
//   a5            D[:, own] = 1/2 (V - X V),  V = S^-1[:, own]            kDensity
//   a4 last iteration folded into a5   U = V + 1/2 E V  (reading 9)                  kLastHalf
//   a2 refinement of the own columns   T = I[:, own] - S V0,  V1 = V0 + A0 T  (reading 11)     kOwnResid, kOwnCorrect
//
// Orientation: C^T = V^T A^T, i.e. the MMA's M side (16) carries the six columns of V twice -- rows 0..5 its FP16 hi
// part, rows 8..13 its lo part * 2^11 -- and the N side (8) rows of A.  A thread loads 16 contiguous bytes (8 rows) of
// four columns k of A (a warp instruction: 4 x 128 contiguous bytes) and pairs the halves of two columns with one
// PRMT into the B fragment of the row's tile; no shared-memory staging of A.  One accumulator tile holds
// c0,c1 = A_hi V_hi and c2,c3 = A_hi V_lo + A_lo V_hi (the second MMA feeds V_hi into rows 8..13), so that
// C = c01 + c23 * 2^-11 has the 22 bits of both operands.
#include "common.cuh"

namespace {

constexpr int kThinThreads = 256;
constexpr int kThinRowWarps = 8;   // warps side by side along the rows of a row block
constexpr int kThinRows = 64 * kThinRowWarps;   // rows of A per row block
constexpr int kThinCtaRows = kThinRows;  // rows per CTA (row blocks one after the other: the staged thin operand serves both)
constexpr int kThinSlices = 8 / kThinRowWarps;     // k slices per CTA, summed through shared memory in a fixed order (run-to-run bitwise equal)

enum ThinMode { kDensity = 0, kLastHalf = 1, kOwnResid = 2, kOwnCorrect = 3, kScaledOut = 4 };

struct ThinArgs {
  const int32_t *row_ptr, *col_idx;
  int mol_begin, ld;
  int64_t slab;
  const __half *a_hi[2], *a_lo[2];   // planes of A by the parity of iters[mat] (iters null: [0]); a_lo null: FP16 A
  const int32_t *iters;
  const float *sinv;                 // FP32 S^-1 (own columns valid), [count][slab]
  const __half *a0;                  // kOwnResid / kOwnCorrect: FP16 approximate inverse
  float *thin;                       // [count][6][ld]: U (kLastHalf out, kDensity in when folded), T (kOwnResid out, kOwnCorrect in)
  int folded;                        // kDensity: V is U from thin, the diagonal gets the pending half iteration
  const __half *e_hi, *e_lo;         // kDensity, folded: E_k for the diagonal
  float *d_val;                      // kDensity: column-owned block store
  double *ne_diag;                   // kDensity: sum of 1 - X_rr over the own rows, or null
  float *out32;                      // kOwnCorrect: FP32 S^-1, own columns written
  float *thin_out;                   // kDensity: when set, 1/2 (V - X V) goes to this [count][6][ld] scratch instead of d_val
  const float *scale;                // kScaledOut: d_val = (A thin) / scale[mat]  (Loewdin form: D[:, own] = Z U / s_S)
  int v32;                           // kOwnResid / kOwnCorrect: the current V is in the own columns of sinv (a later
                                     // refinement round) instead of being A0's own columns
};

__device__ __forceinline__ uint32_t pack_half2(float a, float b) {
  const __half2 h = __floats2half2_rn(a, b);
  return *reinterpret_cast<const uint32_t *>(&h);
}
__device__ __forceinline__ void mma16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                         uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// eight rows (16 bytes) of column k of a plane, zero beyond column n
__device__ __forceinline__ uint4 load_rows8(const __half *plane, int64_t off, bool ok) {
  return ok ? __ldg(reinterpret_cast<const uint4 *>(plane + off)) : make_uint4(0u, 0u, 0u, 0u);
}
__device__ __forceinline__ float split_at(const __half *hi, const __half *lo, int64_t off) {
  float v = __half2float(hi[off]);
  if (lo) v = fmaf(__half2float(lo[off]), 1.f / 2048.f, v);
  return v;
}

// the eight row tiles of one 16-column step: q[j] = 8 rows of columns k0 + 2t + {0, 1, 8, 9}
template <bool kLoPlane>
__device__ __forceinline__ void step_mma(float (&acc)[8][4], const uint4 (&q)[4], const uint4 &f) {
  const uint32_t w0[4] = {q[0].x, q[0].y, q[0].z, q[0].w}, w1[4] = {q[1].x, q[1].y, q[1].z, q[1].w};
  const uint32_t w2[4] = {q[2].x, q[2].y, q[2].z, q[2].w}, w3[4] = {q[3].x, q[3].y, q[3].z, q[3].w};
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const uint32_t sel = (i & 1) ? 0x7632u : 0x5410u;
    const uint32_t b0 = __byte_perm(w0[i >> 1], w1[i >> 1], sel), b1 = __byte_perm(w2[i >> 1], w3[i >> 1], sel);
    if constexpr (kLoPlane) mma16816(acc[i], 0u, f.x, 0u, f.z, b0, b1);   // V_hi in rows 8..13: A_lo V_hi joins A_hi V_lo
    else mma16816(acc[i], f.x, f.y, f.z, f.w, b0, b1);
  }
}

template <int kMode, bool kLo>
__global__ void __launch_bounds__(kThinThreads, 2) k_thin_mma(const ThinArgs a) {
  // register stages of A in flight per thread: 16 bytes x 4 columns [x 2 planes] each
  constexpr int kDepth = kLo ? 2 : 4;
  extern __shared__ __align__(16) uint8_t smem_raw[];
  const int mat = blockIdx.y;
  const int j = a.mol_begin + mat;
  const int lo = a.row_ptr[j];
  const int m = a.row_ptr[j + 1] - lo;
  const int n = m * NOLSM_BS;
  if ((int)blockIdx.x * kThinCtaRows >= n) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t = lane & 3;
  const int ld = a.ld;
  const int nkb = (n + 15) >> 4;                              // 16-column steps
  uint4 *s_frag = reinterpret_cast<uint4 *>(smem_raw);        // [nkb][6][4]: A fragments of the stacked V^T
  float *s_red = reinterpret_cast<float *>(s_frag + (size_t)nkb * 24);   // [kThinSlices][kThinRows][6]
  const int par = a.iters ? (a.iters[mat] & 1) : 0;
  const __half *ahi = a.a_hi[par] + (int64_t)mat * a.slab;
  const __half *alo = kLo ? a.a_lo[par] + (int64_t)mat * a.slab : nullptr;
  const float *sj = a.sinv ? a.sinv + (int64_t)mat * a.slab : nullptr;
  const __half *a0j = a.a0 ? a.a0 + (int64_t)mat * a.slab : nullptr;
  float *tj = a.thin ? a.thin + (int64_t)mat * NOLSM_BS * ld : nullptr;

  const int rw = (warp % kThinRowWarps) * 64;                 // this warp's rows inside a row block
  const int ks = warp / kThinRowWarps;
  const int per = (nkb + kThinSlices - 1) / kThinSlices;
  const int kb0 = ks * per, kb1 = min(nkb, kb0 + per);
  uint4 qh[kDepth][4], ql[kLo ? kDepth : 1][4];
  auto fetch = [&](int kb, int r0, uint4 (&h)[4], uint4 (&l)[4]) {
    const int k = kb * 16 + 2 * t;
    const int kk[4] = {k, k + 1, k + 8, k + 9};
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int64_t off = (int64_t)kk[e] * ld + r0 + 8 * g;
      h[e] = load_rows8(ahi, off, kk[e] < n);
      if constexpr (kLo) l[e] = load_rows8(alo, off, kk[e] < n);
    }
  };
  auto prologue = [&](int r0) {
    if (r0 < n) {
#pragma unroll
      for (int sg = 0; sg < kDepth - 1; ++sg)
        if (kb0 + sg < kb1) fetch(kb0 + sg, r0, qh[sg], ql[kLo ? sg : 0]);
    }
  };
  const int rb_first = blockIdx.x * kThinCtaRows;
  prologue(rb_first + rw);   // the first loads of A are under way while the thin operand is staged

  // position of j in its own (sorted) neighbour list = entries below j.  All loads of this kernel's prologue and
  // epilogue are issued in batches: under the streaming load of the other CTAs a dependent round trip costs
  // microseconds, and a CTA only streams for a few tens of them.
  int own0 = 0;
  for (int base = 0; base < m; base += 8 * 32) {
    int c[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int i = base + 32 * u + lane;
      c[u] = i < m ? a.col_idx[lo + i] : j;
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) own0 += c[u] < j ? 1 : 0;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) own0 += __shfl_xor_sync(0xffffffffu, own0, d);
  own0 *= NOLSM_BS;
  // elements (k, p), (k + 1, p) of the thin operand, k even
  auto vsrc2 = [&](int k, int p) -> float2 {
    if (k >= n) return make_float2(0.f, 0.f);
    if constexpr (kMode == kOwnResid) {
      if (a.v32) return *reinterpret_cast<const float2 *>(sj + (int64_t)(own0 + p) * ld + k);
      return __half22float2(*reinterpret_cast<const __half2 *>(a0j + (int64_t)(own0 + p) * ld + k));
    } else {
      const float *src = (kMode == kOwnCorrect || kMode == kScaledOut || (kMode == kDensity && a.folded)) ? tj + (int64_t)p * ld
                                                                                  : sj + (int64_t)(own0 + p) * ld;
      return *reinterpret_cast<const float2 *>(src + k);
    }
  };
  // item = (p, pair of columns): one half (hi, lo words) of the fragment of thread t of step kb
  const int pairs = nkb * 8;
  for (int base = threadIdx.x; base < NOLSM_BS * pairs; base += 4 * kThinThreads) {
    float2 v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = base + u * kThinThreads;
      v[u] = i < NOLSM_BS * pairs ? vsrc2(2 * (i % pairs), i / pairs) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = base + u * kThinThreads;
      if (i < NOLSM_BS * pairs) {
        const int p = i / pairs, kp = i - p * pairs;
        const int kb = kp >> 3, tt = kp & 3, upper = (kp >> 2) & 1;
        const float l0 = (v[u].x - __half2float(__float2half_rn(v[u].x))) * 2048.f;
        const float l1 = (v[u].y - __half2float(__float2half_rn(v[u].y))) * 2048.f;
        reinterpret_cast<uint2 *>(s_frag + (kb * 6 + p) * 4 + tt)[upper] = make_uint2(pack_half2(v[u].x, v[u].y), pack_half2(l0, l1));
      }
    }
  }
  __syncthreads();

  for (int rb = rb_first; rb < min(n, rb_first + kThinCtaRows); rb += kThinRows) {
    const int r0 = rb + rw;
    if (rb != rb_first) prologue(r0);
    float acc[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.f;
    if (r0 < n) {
      for (int kb = kb0; kb < kb1; kb += kDepth) {
#pragma unroll
        for (int sg = 0; sg < kDepth; ++sg) {
          if (kb + sg < kb1) {
            constexpr int kAhead = kDepth - 1;
            if (kb + sg + kAhead < kb1)
              fetch(kb + sg + kAhead, r0, qh[(sg + kAhead) % kDepth], ql[kLo ? (sg + kAhead) % kDepth : 0]);
            uint4 f = make_uint4(0u, 0u, 0u, 0u);
            if (g < NOLSM_BS) f = s_frag[((kb + sg) * 6 + g) * 4 + t];
            step_mma<false>(acc, qh[sg], f);
            if constexpr (kLo) step_mma<true>(acc, ql[sg], f);
          }
        }
      }
    }
    if (g < NOLSM_BS) {   // C^T rows 0..5 (hi) and 8..13 (lo * 2^11) of column p = g; tile i holds rows r0 + 8 n + i
      float *red = s_red + (size_t)ks * kThinRows * NOLSM_BS;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        red[(rw + 16 * t + i) * NOLSM_BS + g] = fmaf(acc[i][2], 1.f / 2048.f, acc[i][0]);
        red[(rw + 16 * t + 8 + i) * NOLSM_BS + g] = fmaf(acc[i][3], 1.f / 2048.f, acc[i][1]);
      }
    }
    __syncthreads();
    auto total = [&](int i) {   // i = row * 6 + p
      float c = s_red[i];
#pragma unroll
      for (int sl = 1; sl < kThinSlices; ++sl) c += s_red[sl * kThinRows * NOLSM_BS + i];
      return c;
    };
    static_assert(kThinRows * NOLSM_BS % (4 * kThinThreads) == 0, "finalize: four outputs per thread and pass");
    for (int base = threadIdx.x; base < kThinRows * NOLSM_BS; base += 4 * kThinThreads) {
      float v[4];
      int rr[4], pp[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = base + u * kThinThreads;
        if constexpr (kMode == kDensity || kMode == kScaledOut) { rr[u] = i / NOLSM_BS; pp[u] = i - rr[u] * NOLSM_BS; }   // [n][6] block column of D
        else { pp[u] = i / kThinRows; rr[u] = i - pp[u] * kThinRows; }                              // [6][ld] thin / dense columns
        const int r = rb + rr[u];
        v[u] = 0.f;
        if (r < n) {
          if constexpr (kMode == kDensity || kMode == kLastHalf) v[u] = sj[(int64_t)(own0 + pp[u]) * ld + r];
          else if constexpr (kMode == kOwnCorrect)
            v[u] = a.v32 ? sj[(int64_t)(own0 + pp[u]) * ld + r] : __half2float(a0j[(int64_t)(own0 + pp[u]) * ld + r]);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = rb + rr[u], p = pp[u];
        if (r >= n) continue;
        const float c = total(rr[u] * NOLSM_BS + p);
        if constexpr (kMode == kDensity) {
          if (a.thin_out) a.thin_out[((int64_t)mat * NOLSM_BS + p) * ld + r] = 0.5f * (v[u] - c);
          else a.d_val[(int64_t)lo * 36 + (int64_t)r * NOLSM_BS + p] = 0.5f * (v[u] - c);
        } else if constexpr (kMode == kScaledOut) {
          a.d_val[(int64_t)lo * 36 + (int64_t)r * NOLSM_BS + p] = c / a.scale[mat];
        }
        else if constexpr (kMode == kLastHalf) tj[(int64_t)p * ld + r] = fmaf(0.5f, c, v[u]);
        else if constexpr (kMode == kOwnResid) tj[(int64_t)p * ld + r] = (r == own0 + p ? 1.f : 0.f) - c;
        else a.out32[(int64_t)mat * a.slab + (int64_t)(own0 + p) * ld + r] = v[u] + c;
      }
    }
    __syncthreads();   // s_red is rewritten by the next row block
  }
  if constexpr (kMode == kDensity) {
    if (a.ne_diag != nullptr && blockIdx.x == 0 && warp < NOLSM_BS) {
      // electron count: 1 - X_rr over the own rows; folded: the diagonal of X_{k+1} = X_k + 1/2 X_k E_k
      const int r = own0 + warp;
      float dot = 0.f;
      if (a.folded) {
        const int64_t eoff = (int64_t)mat * a.slab + (int64_t)r * ld;
        for (int k = lane; k < n; k += 32)
          dot = fmaf(split_at(ahi, alo, (int64_t)k * ld + r), split_at(a.e_hi + eoff, a.e_lo ? a.e_lo + eoff : nullptr, k), dot);
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, d);
      }
      if (lane == 0) atomicAdd(a.ne_diag, (double)(1.f - fmaf(0.5f, dot, split_at(ahi, alo, (int64_t)r * ld + r))));
    }
  }
}

template <int kMode>
cudaError_t thin_launch(const nolsm_batch *b, const ThinArgs &a, cudaStream_t st) {
  const int nkb = (b->max_n + 15) / 16;
  const size_t smem = (size_t)nkb * 24 * sizeof(uint4) + (size_t)kThinSlices * kThinRows * NOLSM_BS * sizeof(float);
  if (smem > 200 * 1024) return cudaErrorInvalidValue;   // the thin operand of one submatrix must fit in shared memory
  const bool lo = a.a_lo[0] != nullptr;
  if (smem > 48 * 1024) {   // per device and cheap: set on every such launch (a process may use several devices)
    cudaError_t e = lo ? cudaFuncSetAttribute(k_thin_mma<kMode, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                       : cudaFuncSetAttribute(k_thin_mma<kMode, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  dim3 grid((b->max_n + kThinCtaRows - 1) / kThinCtaRows, b->count);
  if (lo) k_thin_mma<kMode, true><<<grid, kThinThreads, smem, st>>>(a);
  else k_thin_mma<kMode, false><<<grid, kThinThreads, smem, st>>>(a);
  return cudaGetLastError();
}

ThinArgs base_args(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx) {
  ThinArgs a;
  memset(&a, 0, sizeof(a));
  a.row_ptr = row_ptr;
  a.col_idx = col_idx;
  a.mol_begin = b->mol_begin;
  a.ld = b->ld;
  a.slab = (int64_t)b->ld * b->ld;
  return a;
}

}  // namespace

// a5 on a split iterate (x.hi0 set).  u_thin set: the last iteration is pending (e_hi [+ e_lo] = E_k): U = V + 1/2 E_k V
// first, then D[:, own] = 1/2 (V - X_k U).
cudaError_t launch_density_split(const nolsm_batch *b, const XRef &x, const float *sinv, const int32_t *row_ptr,
                                 const int32_t *col_idx, float *d_val, double *ne_diag, const __half *e_hi,
                                 const __half *e_lo, float *u_thin, cudaStream_t st, float *thin_out) {
  if (b->count == 0) return cudaSuccess;
  if (u_thin) {
    ThinArgs h = base_args(b, row_ptr, col_idx);
    h.a_hi[0] = h.a_hi[1] = e_hi;
    h.a_lo[0] = h.a_lo[1] = e_lo;
    h.sinv = sinv;
    h.thin = u_thin;
    cudaError_t e = thin_launch<kLastHalf>(b, h, st);
    if (e != cudaSuccess) return e;
  }
  ThinArgs a = base_args(b, row_ptr, col_idx);
  a.a_hi[0] = x.hi0; a.a_hi[1] = x.hi1;
  a.a_lo[0] = x.lo0; a.a_lo[1] = x.lo1;
  a.iters = b->d_iters;
  a.sinv = sinv;
  a.thin = u_thin;
  a.folded = u_thin ? 1 : 0;
  a.e_hi = e_hi;
  a.e_lo = e_lo;
  a.d_val = d_val;
  a.thin_out = thin_out;
  a.ne_diag = ne_diag;
  return thin_launch<kDensity>(b, a, st);
}

// Newton refinement of the six own columns of S^-1 alone (reading 11, own-columns form): with A0 the
// FP16-quality inverse of the Eq. 15-17 iteration and V0 = A0[:, own],  V1 = V0 + A0 (I[:, own] - S V0); the error
// (I - A0 S)(V - V0) is of second order whatever the rounding of A0, as long as both uses read the same A0.
// s_hi, s_lo: split S; thin: scratch of count * 6 * ld floats; out32: FP32 S^-1, its own columns are written.
cudaError_t launch_own_refine(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx, const __half *s_hi,
                              const __half *s_lo, const __half *a0, float *thin, float *out32, int rounds,
                              cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  for (int round = 0; round < rounds; ++round) {   // round r: V_{r+1} = V_r + A0 (I[:, own] - S V_r), error F^(r+2) V
    ThinArgs r = base_args(b, row_ptr, col_idx);
    r.a_hi[0] = r.a_hi[1] = s_hi;
    r.a_lo[0] = r.a_lo[1] = s_lo;
    r.a0 = a0;
    r.thin = thin;
    r.v32 = round > 0 ? 1 : 0;
    r.sinv = round > 0 ? out32 : nullptr;
    cudaError_t e = thin_launch<kOwnResid>(b, r, st);
    if (e != cudaSuccess) return e;
    ThinArgs c = base_args(b, row_ptr, col_idx);
    c.a_hi[0] = c.a_hi[1] = a0;
    c.a0 = a0;
    c.thin = thin;
    c.out32 = out32;
    c.v32 = r.v32;
    c.sinv = r.sinv;
    e = thin_launch<kOwnCorrect>(b, c, st);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

// Loewdin form: D[:, own] = S^-1/2 P S^-1/2[:, own] = Z U / s_S with U = P Z[:, own] in thin_in
// ([count][6][ld]) and Z = (S / s_S)^-1/2 as a split pair; written to the column-owned block store.
cudaError_t launch_scaled_out(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx, const __half *a_hi,
                              const __half *a_lo, float *thin_in, const float *scale, float *d_val, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  ThinArgs a = base_args(b, row_ptr, col_idx);
  a.a_hi[0] = a.a_hi[1] = a_hi;
  a.a_lo[0] = a.a_lo[1] = a_lo;
  a.thin = thin_in;
  a.scale = scale;
  a.d_val = d_val;
  return thin_launch<kScaledOut>(b, a, st);
}
