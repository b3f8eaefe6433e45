// a0 neighbour lists, a1 gather, a1' element generation from positions, a5/a6 density columns + write-back, a7 block trace.
// All integer work is exact (int64 squared distances on the 2^-16 A grid, reading 2).
#include "common.cuh"

// ------------------------------------------------------------------------------------------------
// a0: brute-force neighbour search, one warp per molecule j, candidates i scanned in ascending order
// so the list comes out sorted (Fig. 2 b,c PAPER.md:172,190).  Positions are staged through shared
// memory in tiles so every block reads the position array once per tile, coalesced.
// ------------------------------------------------------------------------------------------------
#define NB_WARPS 8
#define NB_TILE 1024

__device__ __forceinline__ int64_t min_image_sq(int32_t xi, int32_t yi, int32_t zi, int32_t xj,
                                                int32_t yj, int32_t zj, int32_t bx, int32_t by,
                                                int32_t bz) {
  int32_t dx = xi - xj, dy = yi - yj, dz = zi - zj;
  int32_t hx = bx >> 1, hy = by >> 1, hz = bz >> 1;
  if (dx > hx) dx -= bx; else if (dx < -hx) dx += bx;
  if (dy > hy) dy -= by; else if (dy < -hy) dy += by;
  if (dz > hz) dz -= bz; else if (dz < -hz) dz += bz;
  return (int64_t)dx * dx + (int64_t)dy * dy + (int64_t)dz * dz;
}

template <bool FILL>
__global__ void __launch_bounds__(NB_WARPS * 32)
k_neighbours(int n_mol, const int32_t *__restrict__ pos, int32_t bx, int32_t by, int32_t bz,
             int64_t rc2, int32_t *__restrict__ counts, const int32_t *__restrict__ row_ptr,
             int32_t *__restrict__ col_idx) {
  __shared__ int32_t sp[NB_TILE * 3];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int j = blockIdx.x * NB_WARPS + warp;
  const bool live = j < n_mol;
  int32_t xj = 0, yj = 0, zj = 0;
  if (live) { xj = pos[3 * j]; yj = pos[3 * j + 1]; zj = pos[3 * j + 2]; }
  int32_t found = 0;
  int32_t out = (FILL && live) ? row_ptr[j] : 0;
  for (int base = 0; base < n_mol; base += NB_TILE) {
    const int cnt = min(NB_TILE, n_mol - base);
    __syncthreads();
    for (int t = threadIdx.x; t < cnt * 3; t += blockDim.x) sp[t] = pos[(size_t)base * 3 + t];
    __syncthreads();
    if (!live) continue;
    for (int t = 0; t < cnt; t += 32) {
      const int i = t + lane;
      bool ok = false;
      if (i < cnt)
        ok = min_image_sq(sp[3 * i], sp[3 * i + 1], sp[3 * i + 2], xj, yj, zj, bx, by, bz) <= rc2;
      const unsigned m = __ballot_sync(0xffffffffu, ok);
      if (FILL) {
        if (ok) col_idx[out + __popc(m & ((1u << lane) - 1u))] = base + i;
        out += __popc(m);
      } else {
        found += __popc(m);
      }
    }
  }
  if (!FILL && live && lane == 0) counts[j] = found;
}

cudaError_t launch_neighbour_count(int n_mol, const int32_t *pos, const int32_t *box, int32_t rc,
                                   int32_t *counts, cudaStream_t st) {
  if (n_mol <= 0) return cudaSuccess;
  int grid = (n_mol + NB_WARPS - 1) / NB_WARPS;
  k_neighbours<false><<<grid, NB_WARPS * 32, 0, st>>>(n_mol, pos, box[0], box[1], box[2],
                                                      (int64_t)rc * rc, counts, nullptr, nullptr);
  return cudaGetLastError();
}

cudaError_t launch_neighbour_fill(int n_mol, const int32_t *pos, const int32_t *box, int32_t rc,
                                  const int32_t *row_ptr, int32_t *col_idx, cudaStream_t st) {
  if (n_mol <= 0) return cudaSuccess;
  int grid = (n_mol + NB_WARPS - 1) / NB_WARPS;
  k_neighbours<true><<<grid, NB_WARPS * 32, 0, st>>>(n_mol, pos, box[0], box[1], box[2],
                                                     (int64_t)rc * rc, nullptr, row_ptr, col_idx);
  return cudaGetLastError();
}

// Exclusive prefix sum of counts[0..n) into row_ptr[0..n] by one block (n is the number of molecules:
// a few hundred thousand at most, so one block walking the array in 1024-element steps is enough).
__global__ void __launch_bounds__(1024) k_exclusive_scan(const int32_t *__restrict__ counts,
                                                         int32_t *__restrict__ row_ptr, int n) {
  __shared__ int32_t warp_sums[32];
  __shared__ int32_t carry_s;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < n; base += 1024) {
    const int i = base + threadIdx.x;
    int32_t v = i < n ? counts[i] : 0;
    int32_t x = v;
    for (int d = 1; d < 32; d <<= 1) {
      int32_t y = __shfl_up_sync(0xffffffffu, x, d);
      if (lane >= d) x += y;
    }
    if (lane == 31) warp_sums[warp] = x;
    __syncthreads();
    if (warp == 0) {
      int32_t w = warp_sums[lane];
      for (int d = 1; d < 32; d <<= 1) {
        int32_t y = __shfl_up_sync(0xffffffffu, w, d);
        if (lane >= d) w += y;
      }
      warp_sums[lane] = w;
    }
    __syncthreads();
    const int32_t carry = carry_s;
    const int32_t incl = x + (warp > 0 ? warp_sums[warp - 1] : 0) + carry;
    if (i < n) row_ptr[i] = incl - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = incl;
    __syncthreads();
  }
  if (threadIdx.x == 0) row_ptr[n] = carry_s;
}

cudaError_t launch_exclusive_scan(const int32_t *counts, int32_t *row_ptr, int n, cudaStream_t st) {
  k_exclusive_scan<<<1, 1024, 0, st>>>(counts, row_ptr, n);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a1: gather (submatrix construction, step (i) PAPER.md:140, NOLSM PAPER.md:158).
// One warp per block-column b of submatrix j.  For every block-row a the lanes binary-search
// neighbour N_j[b] in the CSR row of neighbour N_j[a]; the hit positions are kept in shared memory.
// Then the six dense columns 6b..6b+5 are written top to bottom, lanes along the rows, so every
// store instruction writes 128 contiguous bytes of the column-major output.  Rows and columns
// between n_j and the tile-padded extent are zero, except a unit diagonal in S (keeps the padded S
// SPD; the padded part decouples exactly).
// ------------------------------------------------------------------------------------------------
#define GA_WARPS 4

// Where a submatrix builder writes: the FP32 matrices and, when the pointers are set, their split FP16
// copies (hi = fp16(v), lo = fp16((v - hi) 2^11): the operands of the FP32-quality products, same
// arithmetic as k_scale_copy) so that no conversion pass has to read the matrices again.
struct BuildOut {
  float *h32, *s32;           // may be null: inside nolsm_solve_mu only the split copies are read
  float *s_norm;              // [2 * count], zeroed by the caller: max absolute column sum of the true n x n part of
                              // T_j(S) (= ||S||_1 = ||S||_inf, S symmetric) in [mat] and [count + mat], or null
  int count;
  __half *h_hi, *h_lo, *s_hi, *s_lo;
};

__device__ __forceinline__ void split_pair(float v0, float v1, __half2 &hi, __half2 &lo) {
  const __half a = __float2half_rn(v0), b = __float2half_rn(v1);
  hi = __halves2half2(a, b);
  lo = __floats2half2_rn((v0 - __half2float(a)) * 2048.f, (v1 - __half2float(b)) * 2048.f);
}

// Rows r, r+1 (r even) of the six columns c0..c0+5: 8-byte FP32 stores (256 bytes per warp instruction)
// and 4-byte FP16 stores (128 bytes per warp instruction).
__device__ __forceinline__ void emit_rows2(const BuildOut &out, int64_t base, int ld, int c0, int r, int P,
                                           const float (&hv)[2][NOLSM_BS], const float (&sv)[2][NOLSM_BS]) {
#pragma unroll
  for (int p = 0; p < NOLSM_BS; ++p) {
    if (c0 + p < P) {
      const int64_t off = base + (int64_t)(c0 + p) * ld + r;
      if (out.h32) *reinterpret_cast<float2 *>(out.h32 + off) = make_float2(hv[0][p], hv[1][p]);
      if (out.s32) *reinterpret_cast<float2 *>(out.s32 + off) = make_float2(sv[0][p], sv[1][p]);
      __half2 hi, lo;
      if (out.h_hi) {
        split_pair(hv[0][p], hv[1][p], hi, lo);
        *reinterpret_cast<__half2 *>(out.h_hi + off) = hi;
        *reinterpret_cast<__half2 *>(out.h_lo + off) = lo;
      }
      if (out.s_hi) {
        split_pair(sv[0][p], sv[1][p], hi, lo);
        *reinterpret_cast<__half2 *>(out.s_hi + off) = hi;
        *reinterpret_cast<__half2 *>(out.s_lo + off) = lo;
      }
    }
  }
}

__global__ void __launch_bounds__(GA_WARPS * 32)
k_gather(const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx,
         const int32_t *__restrict__ list_ptr, const int32_t *__restrict__ list_idx,
         const float *__restrict__ h_val, const float *__restrict__ s_val, int mol_begin, int ld,
         int64_t slab, BuildOut out) {
  // (list_ptr, list_idx): the row set of every submatrix -- the molecule's own neighbour list (= the store's
  // pattern arrays) or the merged row set of a combined submatrix
  extern __shared__ int32_t s_pos[];  // [GA_WARPS][m_max]
  const int mat = blockIdx.y;
  const int j = mol_begin + mat;
  const int lo = list_ptr[j];
  const int m = list_ptr[j + 1] - lo;
  const int n = m * NOLSM_BS;
  const int P = (n + NOLSM_TILE_M - 1) / NOLSM_TILE_M * NOLSM_TILE_M;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m_pad_blocks = (P + NOLSM_BS - 1) / NOLSM_BS;  // block-columns incl. padding
  int32_t *pos = s_pos + warp * ((ld + NOLSM_BS - 1) / NOLSM_BS + 1);
  const int64_t base = (int64_t)mat * slab;
  for (int b = blockIdx.x * GA_WARPS + warp; b < m_pad_blocks; b += gridDim.x * GA_WARPS) {
    if (b < m) {
      const int ib = list_idx[lo + b];
      for (int a = lane; a < m; a += 32) {
        const int ia = list_idx[lo + a];
        int l = row_ptr[ia], r = row_ptr[ia + 1];
        const int end = r;
        while (l < r) {  // lower bound of ib in the sorted CSR row of ia
          const int mid = (l + r) >> 1;
          if (col_idx[mid] < ib) l = mid + 1; else r = mid;
        }
        pos[a] = (l < end && col_idx[l] == ib) ? l : -1;
      }
    }
    __syncwarp();
    // Lane = two consecutive rows (always rows o, o+1 of one block, o even).  What they contribute to this
    // block column are 48 contiguous bytes of the store: three 16-byte loads per matrix.
    const int c0 = b * NOLSM_BS;
    float csum[NOLSM_BS];
#pragma unroll
    for (int p = 0; p < NOLSM_BS; ++p) csum[p] = 0.f;
    for (int r = 2 * lane; r < P; r += 64) {
      float hv[2][NOLSM_BS], sv[2][NOLSM_BS];
#pragma unroll
      for (int p = 0; p < NOLSM_BS; ++p) hv[0][p] = hv[1][p] = sv[0][p] = sv[1][p] = 0.f;
      if (c0 < n && r < n) {
        const int a = r / NOLSM_BS, o = r - a * NOLSM_BS;
        const int k = pos[a];
        if (k >= 0) {
          const float4 *hp = reinterpret_cast<const float4 *>(h_val + (int64_t)k * 36 + o * NOLSM_BS);
          const float4 *sp = reinterpret_cast<const float4 *>(s_val + (int64_t)k * 36 + o * NOLSM_BS);
          const float4 x0 = __ldg(hp), x1 = __ldg(hp + 1), x2 = __ldg(hp + 2);
          const float4 y0 = __ldg(sp), y1 = __ldg(sp + 1), y2 = __ldg(sp + 2);
          hv[0][0] = x0.x; hv[0][1] = x0.y; hv[0][2] = x0.z; hv[0][3] = x0.w; hv[0][4] = x1.x; hv[0][5] = x1.y;
          hv[1][0] = x1.z; hv[1][1] = x1.w; hv[1][2] = x2.x; hv[1][3] = x2.y; hv[1][4] = x2.z; hv[1][5] = x2.w;
          sv[0][0] = y0.x; sv[0][1] = y0.y; sv[0][2] = y0.z; sv[0][3] = y0.w; sv[0][4] = y1.x; sv[0][5] = y1.y;
          sv[1][0] = y1.z; sv[1][1] = y1.w; sv[1][2] = y2.x; sv[1][3] = y2.y; sv[1][4] = y2.z; sv[1][5] = y2.w;
#pragma unroll
          for (int p = 0; p < NOLSM_BS; ++p) csum[p] += fabsf(sv[0][p]) + fabsf(sv[1][p]);
        }
      } else {
#pragma unroll
        for (int p = 0; p < NOLSM_BS; ++p) {   // identity padding of S
          sv[0][p] = (r == c0 + p) ? 1.f : 0.f;
          sv[1][p] = (r + 1 == c0 + p) ? 1.f : 0.f;
        }
      }
      emit_rows2(out, base, ld, c0, r, P, hv, sv);
    }
    if (out.s_norm != nullptr && c0 < n) {   // this warp saw all of its six columns: their absolute sums are complete
      float cmax = 0.f;
#pragma unroll
      for (int p = 0; p < NOLSM_BS; ++p) {
        float v = csum[p];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
        cmax = fmaxf(cmax, v);
      }
      if (lane == 0) {   // non-negative floats order like their bit patterns
        atomicMax(reinterpret_cast<int *>(out.s_norm + mat), __float_as_int(cmax));
        atomicMax(reinterpret_cast<int *>(out.s_norm + out.count + mat), __float_as_int(cmax));
      }
    }
    __syncwarp();
  }
}

static BuildOut build_out(const nolsm_batch *b, float *h_out, float *s_out, bool split_s, float *s_norm = nullptr) {
  BuildOut o;
  o.h32 = h_out;
  o.s32 = s_out;
  o.s_norm = s_norm;
  o.count = b->count;
  o.h_hi = b->h[b->n_half - 2];
  o.h_lo = b->h[b->n_half - 1];
  o.s_hi = split_s ? b->h[b->n_half - 4] : nullptr;
  o.s_lo = split_s ? b->h[b->n_half - 3] : nullptr;
  return o;
}

cudaError_t launch_gather(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx,
                          const int32_t *list_ptr, const int32_t *list_idx,
                          const float *h_val, const float *s_val, float *h_out, float *s_out, bool split_s,
                          float *s_norm, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  const int per_warp = (b->ld + NOLSM_BS - 1) / NOLSM_BS + 1;
  const size_t smem = (size_t)GA_WARPS * per_warp * sizeof(int32_t);
  const int cols = (b->ld + NOLSM_BS - 1) / NOLSM_BS;
  dim3 grid((cols + GA_WARPS - 1) / GA_WARPS, b->count);
  k_gather<<<grid, GA_WARPS * 32, smem, st>>>(row_ptr, col_idx, list_ptr ? list_ptr : row_ptr,
                                              list_idx ? list_idx : col_idx, h_val, s_val, b->mol_begin, b->ld,
                                              (int64_t)b->ld * b->ld, build_out(b, h_out, s_out, split_s, s_norm));
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a1' (SURVEY 8(f)#2; Fig. 2 d-e PAPER.md:172, :202): the elements of T_j(H), T_j(S) evaluated from
// the positions with the two-centre model of nolsm.h (nolsm_model) instead of gathered.  Same shape
// as the gather: one warp per block-column b.  Phase 1: the lanes evaluate, for every block-row a,
// the 3 x 3 site-pair values (two exponentials each) in FP64 -- every operation rounded on its own
// (__dadd_rn/__dmul_rn/...: no contraction into FMAs) in the order nolsm.h states, so the FP32 result
// differs from a host evaluation only where exp()'s last bit does -- and park them in shared memory as
// FP32.  Phase 2 fans them out to the 6 x 6 elements and writes the six columns top to bottom, 128
// contiguous bytes per store instruction.  Whether a pair is stored is the integer minimum-image test
// of a0, so no CSR row of a neighbour is searched.
// ------------------------------------------------------------------------------------------------
struct ModelDev {
  const int32_t *pos;
  int32_t box[3];
  int64_t rc2;
  double unit, len[3], off[3][3];
  double s_ampl, h_ampl, h_len;
  float energy[NOLSM_BS];
  uint32_t site_packed;  // 2 bits per basis function
  int32_t fp32;          // evaluate in FP32 with the SFU exponential instead of FP64
};

__device__ __forceinline__ int32_t wrap_int(int32_t d, int32_t box) {
  const int32_t h = box >> 1;
  return d > h ? d - box : (d < -h ? d + box : d);
}

__device__ __forceinline__ double wrap_axis(double d, double len) {
  return __dsub_rn(d, __dmul_rn(len, rint(__ddiv_rn(d, len))));
}

__global__ void __launch_bounds__(GA_WARPS * 32)
k_generate(const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx,
           const __grid_constant__ ModelDev md, int mol_begin, int ld, int64_t slab, int m_cap, BuildOut out) {
  extern __shared__ float s_gen[];  // [GA_WARPS][2][9 * m_cap]
  const int mat = blockIdx.y;
  const int j = mol_begin + mat;
  const int lo = row_ptr[j];
  const int m = row_ptr[j + 1] - lo;
  const int n = m * NOLSM_BS;
  const int P = (n + NOLSM_TILE_M - 1) / NOLSM_TILE_M * NOLSM_TILE_M;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m_pad_blocks = (P + NOLSM_BS - 1) / NOLSM_BS;
  float *sv9 = s_gen + (size_t)warp * 18 * m_cap;
  float *hv9 = sv9 + 9 * m_cap;
  const int64_t base = (int64_t)mat * slab;
  for (int b = blockIdx.x * GA_WARPS + warp; b < m_pad_blocks; b += gridDim.x * GA_WARPS) {
    if (b < m) {
      const int ib = col_idx[lo + b];
      const int32_t xb = md.pos[3 * ib], yb = md.pos[3 * ib + 1], zb = md.pos[3 * ib + 2];
      for (int t = lane; t < 9 * m; t += 32) {
        const int a = t / 9, q = t - 9 * a;
        const int so = q / 3, sp = q - 3 * so;  // site of the row function, of the column function
        const int ia = col_idx[lo + a];
        const int32_t xa = md.pos[3 * ia], ya = md.pos[3 * ia + 1], za = md.pos[3 * ia + 2];
        float sv = 0.f, hv = 0.f;
        const bool stored = min_image_sq(xa, ya, za, xb, yb, zb, md.box[0], md.box[1], md.box[2]) <= md.rc2;
        if (stored && !(ia == ib && so == sp) && md.fp32) {
          // The paper's choice: FP32 arithmetic, transcendental functions on the special
          // function units.  The centre difference is reduced to its minimum image in integers (exact),
          // the site offsets can push a component past half the box, hence one more wrap.
          const float unit = (float)md.unit;
          float d[3] = {(float)wrap_int(xa - xb, md.box[0]) * unit, (float)wrap_int(ya - yb, md.box[1]) * unit,
                        (float)wrap_int(za - zb, md.box[2]) * unit};
          float r2 = 0.f;
#pragma unroll
          for (int ax = 0; ax < 3; ++ax) {
            const float len = (float)md.len[ax];
            float x = d[ax] + (float)(md.off[so][ax] - md.off[sp][ax]);
            x -= len * rintf(x / len);
            r2 = fmaf(x, x, r2);
          }
          sv = (float)md.s_ampl * __expf(-0.5f * r2);
          hv = (float)md.h_ampl * __expf(-sqrtf(r2) / (float)md.h_len);
        } else if (stored && !(ia == ib && so == sp)) {
          double dx = __dmul_rn((double)(xa - xb), md.unit);
          double dy = __dmul_rn((double)(ya - yb), md.unit);
          double dz = __dmul_rn((double)(za - zb), md.unit);
          dx = wrap_axis(__dsub_rn(__dadd_rn(dx, md.off[so][0]), md.off[sp][0]), md.len[0]);
          dy = wrap_axis(__dsub_rn(__dadd_rn(dy, md.off[so][1]), md.off[sp][1]), md.len[1]);
          dz = wrap_axis(__dsub_rn(__dadd_rn(dz, md.off[so][2]), md.off[sp][2]), md.len[2]);
          const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
          sv = (float)__dmul_rn(md.s_ampl, exp(__dmul_rn(-0.5, r2)));
          hv = (float)__dmul_rn(md.h_ampl, exp(__ddiv_rn(-__dsqrt_rn(r2), md.h_len)));
        }
        sv9[t] = sv;
        hv9[t] = hv;
      }
    }
    __syncwarp();
    const int c0 = b * NOLSM_BS;
    for (int r = 2 * lane; r < P; r += 64) {     // lane = rows o, o+1 of one block (o even), as in k_gather
      float hv[2][NOLSM_BS], sv[2][NOLSM_BS];
      if (c0 < n && r < n) {
        const int a = r / NOLSM_BS, o = r - a * NOLSM_BS;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const int so3 = ((md.site_packed >> (2 * (o + i))) & 3) * 3;
#pragma unroll
          for (int p = 0; p < NOLSM_BS; ++p) {
            if (a == b && o + i == p) {
              sv[i][p] = 1.f;
              hv[i][p] = md.energy[p];
            } else {
              const int k = a * 9 + so3 + ((md.site_packed >> (2 * p)) & 3);
              hv[i][p] = hv9[k];
              sv[i][p] = sv9[k];
            }
          }
        }
      } else {
#pragma unroll
        for (int p = 0; p < NOLSM_BS; ++p) {
          hv[0][p] = hv[1][p] = 0.f;
          sv[0][p] = (r == c0 + p) ? 1.f : 0.f;
          sv[1][p] = (r + 1 == c0 + p) ? 1.f : 0.f;
        }
      }
      emit_rows2(out, base, ld, c0, r, P, hv, sv);
    }
    __syncwarp();
  }
}

cudaError_t launch_generate(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx,
                            const nolsm_model *model, float *h_out, float *s_out, bool split_s,
                            cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  ModelDev md;
  md.pos = model->pos_q;
  md.rc2 = (int64_t)model->rc_q * model->rc_q;
  md.unit = model->unit_per_grid;
  md.site_packed = 0;
  for (int i = 0; i < 3; ++i) {
    md.box[i] = model->box_q[i];
    md.len[i] = (double)model->box_q[i] * model->unit_per_grid;
    for (int k = 0; k < 3; ++k) md.off[i][k] = model->site_offset[i][k];
  }
  for (int o = 0; o < NOLSM_BS; ++o) {
    md.energy[o] = (float)model->orb_energy[o];
    md.site_packed |= (uint32_t)model->orb_site[o] << (2 * o);
  }
  md.s_ampl = model->s_ampl;
  md.h_ampl = model->h_ampl;
  md.h_len = model->h_len;
  md.fp32 = model->eval_fp32;
  const int m_cap = (b->ld + NOLSM_BS - 1) / NOLSM_BS + 1;
  const size_t smem = (size_t)GA_WARPS * 18 * m_cap * sizeof(float);
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(k_generate, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  const int cols = (b->ld + NOLSM_BS - 1) / NOLSM_BS;
  dim3 grid((cols + GA_WARPS - 1) / GA_WARPS, b->count);
  k_generate<<<grid, GA_WARPS * 32, smem, st>>>(row_ptr, col_idx, md, b->mol_begin, b->ld,
                                                (int64_t)b->ld * b->ld, m_cap, build_out(b, h_out, s_out, split_s));
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a5 + a6: D_j[:, own] = 1/2 (I - X_j) S_j^-1[:, own]  (Eq. 12; only the own columns are
// kept) written straight into the column-owned store: rows 6a..6a+5 of the n_j x 6
// result are block (N_j[a], j) = block row_ptr[j]+a of D, so the result is one contiguous run.
// One thread per row r, the six own columns of S^-1 staged in shared memory, X read column by
// column (coalesced).  Also accumulates the diagonal estimate sum_{c in own}(1 - X_cc) (reading 15).
// ------------------------------------------------------------------------------------------------
// Operator cache of nolsm_solve_mu: the true n_j x n_j part of every slab of a batch to / from a dense
// packing (submatrix m at offset sum_{i<m} n_i^2, leading dimension n_m).  grid (count, PK_SPLIT).
#define PK_SPLIT 8
__global__ void __launch_bounds__(256)
k_pack_square(const int32_t *__restrict__ dims, int ld, int64_t slab, float *__restrict__ dense,
              float *__restrict__ packed, int save) {
  __shared__ long long s_part[8];
  __shared__ long long s_off;
  const int m = blockIdx.x;
  long long acc = 0;
  for (int i = threadIdx.x; i < m; i += blockDim.x) acc += (long long)dims[i] * dims[i];
  for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
  if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    long long t = 0;
    for (int w = 0; w < 8; ++w) t += s_part[w];
    s_off = t;
  }
  __syncthreads();
  const int n = dims[m];          // a multiple of 6: rows in pairs
  const int h = n >> 1;
  float2 *pk = reinterpret_cast<float2 *>(packed + s_off);
  float *dj = dense + (int64_t)m * slab;
  const int64_t total = (int64_t)h * n;
  for (int64_t idx = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)PK_SPLIT * blockDim.x) {
    const int c = (int)(idx / h), r2 = (int)(idx - (int64_t)c * h);
    float2 *dp = reinterpret_cast<float2 *>(dj + (int64_t)c * ld) + r2;
    if (save) pk[idx] = *dp; else *dp = pk[idx];
  }
}

cudaError_t launch_pack_square(const nolsm_batch *b, float *dense, float *packed, bool save, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_pack_square<<<dim3(b->count, PK_SPLIT), 256, 0, st>>>(b->d_dims, b->ld, (int64_t)b->ld * b->ld, dense, packed,
                                                          save ? 1 : 0);
  return cudaGetLastError();
}

// Operator cache of nolsm_solve_mu: the six own columns of S_j^-1 to / from a packed [count][6][ld] array.
__global__ void __launch_bounds__(256)
k_own_columns(const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx, int mol_begin, int ld,
              int64_t slab, float *__restrict__ mat, float *__restrict__ packed, int save) {
  const int m_ = blockIdx.x;
  const int j = mol_begin + m_;
  const int lo = row_ptr[j];
  const int m = row_ptr[j + 1] - lo;
  int l = 0, r_ = m;
  while (l < r_) {   // position of j in its own (sorted) neighbour list
    const int mid = (l + r_) >> 1;
    if (col_idx[lo + mid] < j) l = mid + 1; else r_ = mid;
  }
  float *src = mat + (int64_t)m_ * slab + (int64_t)l * NOLSM_BS * ld;   // six consecutive columns
  float *pk = packed + (int64_t)m_ * NOLSM_BS * ld;
  for (int t = threadIdx.x; t < NOLSM_BS * ld; t += blockDim.x) {
    if (save) pk[t] = src[t]; else src[t] = pk[t];
  }
}

cudaError_t launch_own_columns(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx, float *mat,
                               float *packed, bool save, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_own_columns<<<b->count, 256, 0, st>>>(row_ptr, col_idx, b->mol_begin, b->ld, (int64_t)b->ld * b->ld, mat,
                                          packed, save ? 1 : 0);
  return cudaGetLastError();
}

#define DN_THREADS 256

// a5: D columns of the own molecule, 1/2 (V - X V) with V the six own columns of
// S^-1.  An n x n x 6 product bound by reading X once.  CTA = DN_ROWS rows x DN_KSPLIT slices of the k range;
// a thread owns two consecutive rows (n = 6m is even, ld a multiple of 128: every pair is one aligned 4-byte FP16
// or 8-byte FP32 load, so a warp request is a full 128-byte line or two) and one k slice; the slices are summed
// through shared memory.
#define DN_KSPLIT 4
#define DN_ROWS 128   // rows per CTA: (DN_THREADS / DN_KSPLIT) threads x 2 rows
#define DN_RED_FLOATS ((DN_KSPLIT - 1) * DN_ROWS * NOLSM_BS)

__device__ __forceinline__ float2 split_pair(const __half *hi, const __half *lo, int64_t off) {
  const float2 h = __half22float2(__ldg(reinterpret_cast<const __half2 *>(hi + off)));
  if (lo == nullptr) return h;
  const float2 l = __half22float2(__ldg(reinterpret_cast<const __half2 *>(lo + off)));
  return make_float2(fmaf(l.x, 1.f / 2048.f, h.x), fmaf(l.y, 1.f / 2048.f, h.y));
}

// element of the sign iterate: FP32, or hi + lo * 2^-11 (the split master of DESIGN.md reading 12)
template <bool kSplit>
struct XMat {
  const float *x32;
  const __half *hi, *lo;
  __device__ __forceinline__ float at(int64_t off) const {
    if constexpr (kSplit) return fmaf(__half2float(__ldg(lo + off)), 1.f / 2048.f, __half2float(__ldg(hi + off)));
    else return __ldg(x32 + off);
  }
  // elements off, off + 1 (off even)
  __device__ __forceinline__ float2 at2(int64_t off) const {
    if constexpr (kSplit) return split_pair(hi, lo, off);
    else return __ldg(reinterpret_cast<const float2 *>(x32 + off));
  }
};

// position of molecule j in its own (sorted) neighbour list
__device__ __forceinline__ int own_position(const int32_t *__restrict__ col_idx, int lo, int m, int j) {
  int l = 0, r_ = m;
  while (l < r_) {
    const int mid = (l + r_) >> 1;
    if (col_idx[lo + mid] < j) l = mid + 1; else r_ = mid;
  }
  return l;
}

// sum of the k slices: slices 1.. park their partial sums in shared memory, slice 0 adds them up
__device__ __forceinline__ void slice_reduce(float *red, int ks, int rp, float (&acc)[2][NOLSM_BS]) {
  if (ks > 0) {
    float *dst = red + ((ks - 1) * DN_ROWS + 2 * rp) * NOLSM_BS;
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int p = 0; p < NOLSM_BS; ++p) dst[q * NOLSM_BS + p] = acc[q][p];
  }
  __syncthreads();
  if (ks == 0) {
#pragma unroll
    for (int s = 0; s < DN_KSPLIT - 1; ++s) {
      const float *src = red + (s * DN_ROWS + 2 * rp) * NOLSM_BS;
#pragma unroll
      for (int q = 0; q < 2; ++q)
#pragma unroll
        for (int p = 0; p < NOLSM_BS; ++p) acc[q][p] += src[q * NOLSM_BS + p];
    }
  }
}

// acc[q][p] += sum_k A(r + q, k) in(k, p) over k0 <= k < k1: A column by column through load(offset) (rows r, r + 1 as
// one aligned pair, coalesced), row k of the staged thin operand as three broadcast 8-byte loads
template <typename LoadPair>
__device__ __forceinline__ void thin_mac(const float *s_in, int k0, int k1, int ld, int r, LoadPair load,
                                         float (&acc)[2][NOLSM_BS]) {
#pragma unroll 8
  for (int k = k0; k < k1; ++k) {
    const float2 xv = load((int64_t)k * ld + r);
    const float2 *sk = reinterpret_cast<const float2 *>(s_in + k * NOLSM_BS);
    const float2 s0 = sk[0], s1 = sk[1], s2 = sk[2];
    acc[0][0] = fmaf(xv.x, s0.x, acc[0][0]); acc[0][1] = fmaf(xv.x, s0.y, acc[0][1]);
    acc[0][2] = fmaf(xv.x, s1.x, acc[0][2]); acc[0][3] = fmaf(xv.x, s1.y, acc[0][3]);
    acc[0][4] = fmaf(xv.x, s2.x, acc[0][4]); acc[0][5] = fmaf(xv.x, s2.y, acc[0][5]);
    acc[1][0] = fmaf(xv.y, s0.x, acc[1][0]); acc[1][1] = fmaf(xv.y, s0.y, acc[1][1]);
    acc[1][2] = fmaf(xv.y, s1.x, acc[1][2]); acc[1][3] = fmaf(xv.y, s1.y, acc[1][3]);
    acc[1][4] = fmaf(xv.y, s2.x, acc[1][4]); acc[1][5] = fmaf(xv.y, s2.y, acc[1][5]);
  }
}

template <bool kSplit>
__global__ void __launch_bounds__(DN_THREADS)
k_density(const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx, int mol_begin,
          int ld, int64_t slab, const XRef xr,
          const int32_t *__restrict__ iters, const float *__restrict__ sinv,
          const float *__restrict__ u_thin, const __half *__restrict__ e_hi, const __half *__restrict__ e_lo,
          float *__restrict__ d_val, double *__restrict__ ne_diag) {
  // [n][6], row k contiguous: the six own columns V of S^-1, or (u_thin set: last iteration folded in,
  // thin_kernels.cu kLastHalf) U = V + 1/2 E V, so that X U = X_{k+1} V; then the slice sums
  extern __shared__ __align__(16) float s_sinv[];
  const int mat = blockIdx.y;
  const int j = mol_begin + mat;
  const int lo = row_ptr[j];
  const int m = row_ptr[j + 1] - lo;
  const int n = m * NOLSM_BS;
  if ((int)blockIdx.x * DN_ROWS >= n) return;
  const int own0 = own_position(col_idx, lo, m, j) * NOLSM_BS;
  XMat<kSplit> xj;
  if constexpr (kSplit) {
    xj.hi = ((iters[mat] & 1) ? xr.hi1 : xr.hi0) + (int64_t)mat * slab;
    xj.lo = ((iters[mat] & 1) ? xr.lo1 : xr.lo0) + (int64_t)mat * slab;
  } else {
    xj.x32 = xr.x32 + (int64_t)mat * slab;
  }
  const float *sj = sinv + (int64_t)mat * slab;
  const float *uj = u_thin ? u_thin + (int64_t)mat * NOLSM_BS * ld : nullptr;
  for (int t = threadIdx.x; t < NOLSM_BS * n; t += blockDim.x) {
    const int p = t / n, k = t - p * n;
    s_sinv[k * NOLSM_BS + p] = uj ? uj[(int64_t)p * ld + k] : sj[(int64_t)(own0 + p) * ld + k];
  }
  float *red = s_sinv + NOLSM_BS * n;
  __syncthreads();
  const int ks = threadIdx.x / (DN_THREADS / DN_KSPLIT);
  const int rp = threadIdx.x % (DN_THREADS / DN_KSPLIT);
  const int r = blockIdx.x * DN_ROWS + 2 * rp;
  const int klen = (n + DN_KSPLIT - 1) / DN_KSPLIT;
  const int k0 = ks * klen, k1 = min(n, k0 + klen);
  const bool live = r < n;
  float acc[2][NOLSM_BS];
#pragma unroll
  for (int p = 0; p < NOLSM_BS; ++p) acc[0][p] = acc[1][p] = 0.f;
  if (live) thin_mac(s_sinv, k0, k1, ld, r, [&](int64_t off) { return xj.at2(off); }, acc);
  if (live && ne_diag != nullptr && r >= own0 && r < own0 + NOLSM_BS) {
    // electron count: 1 - X_rr of the own rows; with the last iteration folded in, the diagonal of
    // X_{k+1} = X_k + 1/2 X_k E_k, this thread's k slice of the two dot products
    float part = 0.f;
    if (ks == 0) part = 2.f - xj.at((int64_t)r * ld + r) - xj.at((int64_t)(r + 1) * ld + r + 1);
    if (uj) {
      const int64_t eoff = (int64_t)mat * slab + (int64_t)r * ld;
      float dot = 0.f;
      for (int k = k0; k < k1; ++k) {
        float ea = __half2float(e_hi[eoff + k]), eb = __half2float(e_hi[eoff + ld + k]);
        if (e_lo) {
          ea = fmaf(__half2float(e_lo[eoff + k]), 1.f / 2048.f, ea);
          eb = fmaf(__half2float(e_lo[eoff + ld + k]), 1.f / 2048.f, eb);
        }
        const float2 xv = xj.at2((int64_t)k * ld + r);
        dot = fmaf(xv.x, ea, dot);
        dot = fmaf(xv.y, eb, dot);
      }
      part = fmaf(-0.5f, dot, part);
    }
    atomicAdd(ne_diag, (double)part);
  }
  slice_reduce(red, ks, rp, acc);
  if (live && ks == 0) {
    float o[2 * NOLSM_BS];
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int p = 0; p < NOLSM_BS; ++p) {
        const float v = uj ? sj[(int64_t)(own0 + p) * ld + r + q] : s_sinv[(r + q) * NOLSM_BS + p];
        o[q * NOLSM_BS + p] = 0.5f * (v - acc[q][p]);
      }
    // rows r, r + 1 of the [n][6] block column: 12 consecutive floats, 48-byte aligned (r even)
    float4 *out = reinterpret_cast<float4 *>(d_val + ((int64_t)lo * 36 + (int64_t)r * NOLSM_BS));
    out[0] = make_float4(o[0], o[1], o[2], o[3]);
    out[1] = make_float4(o[4], o[5], o[6], o[7]);
    out[2] = make_float4(o[8], o[9], o[10], o[11]);
  }
}

// FP32 copy of a split iterate (for the consumers that read X as FP32: energy products, nolsm_batch_read)
__global__ void __launch_bounds__(256)
k_join_split(const int32_t *__restrict__ dims, const int32_t *__restrict__ iters, int ld, int64_t slab, const XRef xr,
             float *__restrict__ dst) {
  const int mat = blockIdx.y;
  const int n = dims[mat];
  const int P = (n + 3) & ~3;
  const int64_t per = (int64_t)(P >> 2) * n;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= per) return;
  const int c = (int)(i / (P >> 2)), r = (int)(i % (P >> 2)) * 4;
  const int64_t off = (int64_t)mat * slab + (int64_t)c * ld + r;
  const __half *hi = ((iters[mat] & 1) ? xr.hi1 : xr.hi0) + off;
  const __half *lo = ((iters[mat] & 1) ? xr.lo1 : xr.lo0) + off;
  float v[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) v[k] = fmaf(__half2float(lo[k]), 1.f / 2048.f, __half2float(hi[k]));
  *reinterpret_cast<float4 *>(dst + off) = make_float4(v[0], v[1], v[2], v[3]);
}

__global__ void __launch_bounds__(256)
k_own_join(const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx, int mol_begin, int ld, int64_t slab,
           const __half *__restrict__ hi, const __half *__restrict__ lo, float *__restrict__ dst) {
  const int mat = blockIdx.x;
  const int j = mol_begin + mat;
  const int lo_ = row_ptr[j];
  const int m = row_ptr[j + 1] - lo_;
  const int n = m * NOLSM_BS;
  int l = 0, r_ = m;
  while (l < r_) {
    const int mid = (l + r_) >> 1;
    if (col_idx[lo_ + mid] < j) l = mid + 1; else r_ = mid;
  }
  const int own0 = l * NOLSM_BS;
  for (int t = threadIdx.x; t < NOLSM_BS * n; t += blockDim.x) {
    const int p = t / n, k = t - p * n;
    const int64_t off = (int64_t)mat * slab + (int64_t)(own0 + p) * ld + k;
    dst[off] = fmaf(__half2float(lo[off]), 1.f / 2048.f, __half2float(hi[off]));
  }
}

cudaError_t launch_own_join(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx, const __half *hi,
                            const __half *lo, float *dst32, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_own_join<<<b->count, 256, 0, st>>>(row_ptr, col_idx, b->mol_begin, b->ld, (int64_t)b->ld * b->ld, hi, lo, dst32);
  return cudaGetLastError();
}

cudaError_t launch_join_split(const nolsm_batch *b, const XRef &x, float *dst32, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  const int P = (b->max_n + 3) & ~3;
  dim3 grid((unsigned)(((int64_t)(P >> 2) * b->max_n + 255) / 256), (unsigned)b->count);
  k_join_split<<<grid, 256, 0, st>>>(b->d_dims, b->d_iters, b->ld, (int64_t)b->ld * b->ld, x, dst32);
  return cudaGetLastError();
}

cudaError_t launch_density(const nolsm_batch *b, const XRef &x, const float *sinv,
                           const int32_t *row_ptr, const int32_t *col_idx, float *d_val,
                           double *ne_diag, const __half *e_hi, const __half *e_lo, float *u_thin,
                           cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  if (x.hi0)   // split iterate of the tensor-core engine: thin_kernels.cu
    return launch_density_split(b, x, sinv, row_ptr, col_idx, d_val, ne_diag, e_hi, e_lo, u_thin, st);
  if (u_thin) return cudaErrorInvalidValue;   // a pending last iteration only exists on the split iterate
  const size_t smem = ((size_t)NOLSM_BS * b->max_n + DN_RED_FLOATS) * sizeof(float);
  if (smem > 200 * 1024) return cudaErrorInvalidValue;   // six columns of one submatrix must fit in shared memory
  if (smem > 48 * 1024) {   // per device and cheap: set on every such launch (a process may use several devices)
    cudaError_t e = cudaFuncSetAttribute(k_density<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  dim3 grid((b->max_n + DN_ROWS - 1) / DN_ROWS, b->count);
  k_density<false><<<grid, DN_THREADS, smem, st>>>(row_ptr, col_idx, b->mol_begin, b->ld, (int64_t)b->ld * b->ld, x,
                                                   b->d_iters, sinv, nullptr, nullptr, nullptr, d_val, ne_diag);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Block store on a larger pattern (the merged H0 u S pattern): block k of row i of the destination is
// the source's block (i, col_idx_dst[k]) if the source stores that pair, else zero.  One warp per destination block.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_expand_store(int n_mol, const int32_t *__restrict__ rp_src, const int32_t *__restrict__ ci_src,
               const float *__restrict__ val_src, const int32_t *__restrict__ rp_dst,
               const int32_t *__restrict__ ci_dst, float *__restrict__ val_dst) {
  const int lane = threadIdx.x & 31;
  const int i = blockIdx.x;
  if (i >= n_mol) return;
  const int s0 = rp_src[i], sm = rp_src[i + 1] - s0;
  for (int k = rp_dst[i] + (threadIdx.x >> 5); k < rp_dst[i + 1]; k += blockDim.x >> 5) {
    const int c = ci_dst[k];
    int l = 0, r = sm;
    while (l < r) {
      const int mid = (l + r) >> 1;
      if (ci_src[s0 + mid] < c) l = mid + 1; else r = mid;
    }
    const bool hit = l < sm && ci_src[s0 + l] == c;
    for (int e = lane; e < 36; e += 32) val_dst[(int64_t)k * 36 + e] = hit ? val_src[(int64_t)(s0 + l) * 36 + e] : 0.f;
  }
}

cudaError_t launch_expand_store(int n_mol, const int32_t *rp_src, const int32_t *ci_src, const float *val_src,
                                const int32_t *rp_dst, const int32_t *ci_dst, float *val_dst, cudaStream_t st) {
  if (n_mol == 0) return cudaSuccess;
  k_expand_store<<<n_mol, 256, 0, st>>>(n_mol, rp_src, ci_src, val_src, rp_dst, ci_dst, val_dst);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Combined submatrices: one submatrix serves several molecules (its owners).
// Group g has the merged row set U_g = list_idx[list_ptr[g] ..) and the owners own_idx[own_ptr[g] ..).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int lower_bound_i32(const int32_t *a, int n, int key) {
  int l = 0, r = n;
  while (l < r) {
    const int mid = (l + r) >> 1;
    if (a[mid] < key) l = mid + 1; else r = mid;
  }
  return l;
}

// own columns (all owners) of a split matrix to FP32
__global__ void __launch_bounds__(256)
k_own_join_grouped(const int32_t *__restrict__ own_ptr, const int32_t *__restrict__ own_idx,
                   const int32_t *__restrict__ list_ptr, const int32_t *__restrict__ list_idx, int grp_begin, int ld,
                   int64_t slab, const __half *__restrict__ hi, const __half *__restrict__ lo, float *__restrict__ dst) {
  const int mat = blockIdx.x;
  const int g = grp_begin + mat;
  const int l0 = list_ptr[g];
  const int m = list_ptr[g + 1] - l0;
  const int n = m * NOLSM_BS;
  for (int o = own_ptr[g]; o < own_ptr[g + 1]; ++o) {
    const int own0 = lower_bound_i32(list_idx + l0, m, own_idx[o]) * NOLSM_BS;
    for (int t = threadIdx.x; t < NOLSM_BS * n; t += blockDim.x) {
      const int p = t / n, k = t - p * n;
      const int64_t off = (int64_t)mat * slab + (int64_t)(own0 + p) * ld + k;
      dst[off] = fmaf(__half2float(lo[off]), 1.f / 2048.f, __half2float(hi[off]));
    }
  }
}

cudaError_t launch_own_join_grouped(const nolsm_batch *b, const __half *hi, const __half *lo, float *dst32,
                                    cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_own_join_grouped<<<b->count, 256, 0, st>>>(b->g_own_ptr, b->g_own_idx, b->g_list_ptr, b->g_list_idx, b->mol_begin,
                                               b->ld, (int64_t)b->ld * b->ld, hi, lo, dst32);
  return cudaGetLastError();
}

// a5 + a6 for a combined submatrix: for every owner j the columns D[:, own_j] = 1/2 (I - X) S^-1[:, own_j]; the row
// block of molecule i = U[r / 6] goes to block D(i, j) of the column-owned store if i is in N_j (position found in
// the store's pattern), else it is not stored (the result keeps the input pattern).
template <bool kSplit>
__global__ void __launch_bounds__(DN_THREADS)
k_density_grouped(const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx,
                  const int32_t *__restrict__ own_ptr, const int32_t *__restrict__ own_idx,
                  const int32_t *__restrict__ list_ptr, const int32_t *__restrict__ list_idx, int grp_begin, int ld,
                  int64_t slab, const XRef xr, const int32_t *__restrict__ iters, const float *__restrict__ sinv,
                  float *__restrict__ d_val) {
  extern __shared__ __align__(16) float s_sinv[];   // [n][6]: own columns of S^-1 of the current owner
  const int mat = blockIdx.y;
  const int g = grp_begin + mat;
  const int l0 = list_ptr[g];
  const int m = list_ptr[g + 1] - l0;
  const int n = m * NOLSM_BS;
  XMat<kSplit> xj;
  if constexpr (kSplit) {
    xj.hi = ((iters[mat] & 1) ? xr.hi1 : xr.hi0) + (int64_t)mat * slab;
    xj.lo = ((iters[mat] & 1) ? xr.lo1 : xr.lo0) + (int64_t)mat * slab;
  } else {
    xj.x32 = xr.x32 + (int64_t)mat * slab;
  }
  const float *sj = sinv + (int64_t)mat * slab;
  const int r = blockIdx.x * DN_THREADS + threadIdx.x;
  for (int o = own_ptr[g]; o < own_ptr[g + 1]; ++o) {
    const int j = own_idx[o];
    const int own0 = lower_bound_i32(list_idx + l0, m, j) * NOLSM_BS;
    __syncthreads();
    for (int t = threadIdx.x; t < NOLSM_BS * n; t += blockDim.x) {
      const int p = t / n, k = t - p * n;
      s_sinv[k * NOLSM_BS + p] = sj[(int64_t)(own0 + p) * ld + k];
    }
    __syncthreads();
    if (r < n) {
      float acc[NOLSM_BS];
#pragma unroll
      for (int p = 0; p < NOLSM_BS; ++p) acc[p] = 0.f;
#pragma unroll 4
      for (int k = 0; k < n; ++k) {
        const float xv = xj.at((int64_t)k * ld + r);
#pragma unroll
        for (int p = 0; p < NOLSM_BS; ++p) acc[p] = fmaf(xv, s_sinv[k * NOLSM_BS + p], acc[p]);
      }
      const int i = list_idx[l0 + r / NOLSM_BS];
      const int jlo = row_ptr[j], jm = row_ptr[j + 1] - jlo;
      const int q = lower_bound_i32(col_idx + jlo, jm, i);
      if (q < jm && col_idx[jlo + q] == i) {
        float *out = d_val + ((int64_t)(jlo + q) * 36 + (int64_t)(r % NOLSM_BS) * NOLSM_BS);
#pragma unroll
        for (int p = 0; p < NOLSM_BS; ++p) out[p] = 0.5f * (s_sinv[r * NOLSM_BS + p] - acc[p]);
      }
    }
  }
}

cudaError_t launch_density_grouped(const nolsm_batch *b, const XRef &x, const float *sinv, const int32_t *row_ptr,
                                   const int32_t *col_idx, float *d_val, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  const size_t smem = (size_t)NOLSM_BS * b->max_n * sizeof(float);
  if (smem > 200 * 1024) return cudaErrorInvalidValue;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(k_density_grouped<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(k_density_grouped<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  dim3 grid((b->max_n + DN_THREADS - 1) / DN_THREADS, b->count);
  if (x.hi0)
    k_density_grouped<true><<<grid, DN_THREADS, smem, st>>>(row_ptr, col_idx, b->g_own_ptr, b->g_own_idx, b->g_list_ptr,
                                                            b->g_list_idx, b->mol_begin, b->ld, (int64_t)b->ld * b->ld, x,
                                                            b->d_iters, sinv, d_val);
  else
    k_density_grouped<false><<<grid, DN_THREADS, smem, st>>>(row_ptr, col_idx, b->g_own_ptr, b->g_own_idx, b->g_list_ptr,
                                                             b->g_list_idx, b->mol_begin, b->ld, (int64_t)b->ld * b->ld, x,
                                                             b->d_iters, sinv, d_val);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a7: N = 2 sum over stored blocks <D(i,j), S(i,j)>_F  (reading 15).
// One warp per molecule j; lane k handles block (N_j[k], j): D block k of row j against S block
// (i, j), found by binary search of j in row i of S.  FP32 products, FP64 accumulation.
// ------------------------------------------------------------------------------------------------
#define TR_WARPS 4

__global__ void __launch_bounds__(TR_WARPS * 32)
k_trace(const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx, int mol_begin,
        int count, const int32_t *__restrict__ mol_list, const float *__restrict__ d_val,
        const float *__restrict__ s_val, double *__restrict__ ne, double *__restrict__ q_mol) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int mat = blockIdx.x * TR_WARPS + warp;
  if (mat >= count) return;
  const int j = mol_list ? mol_list[mol_begin + mat] : mol_begin + mat;   // owners of combined submatrices: a list
  const int lo = row_ptr[j], hi = row_ptr[j + 1];
  double sum = 0.0;
  for (int k = lo + lane; k < hi; k += 32) {
    const int i = col_idx[k];
    int l = row_ptr[i], r = row_ptr[i + 1];
    const int end = r;
    while (l < r) {
      const int mid = (l + r) >> 1;
      if (col_idx[mid] < j) l = mid + 1; else r = mid;
    }
    if (l < end && col_idx[l] == j) {
      const float *db = d_val + (int64_t)k * 36;
      const float *sb = s_val + (int64_t)l * 36;
      double part = 0.0;
#pragma unroll 4
      for (int e = 0; e < 36; ++e) part += (double)(db[e] * sb[e]);
      sum += part;
    }
  }
  for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
  if (lane == 0) {
    if (q_mol != nullptr) q_mol[j] = 2.0 * sum;
    atomicAdd(ne, 2.0 * sum);
  }
}

cudaError_t launch_trace(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx,
                         const float *d_val, const float *s_val, double *ne, double *q_mol,
                         cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  if (b->grouped) {   // the owners of the batch's groups are own_idx[own_first, own_first + own_count)
    if (b->own_count == 0) return cudaSuccess;
    k_trace<<<(b->own_count + TR_WARPS - 1) / TR_WARPS, TR_WARPS * 32, 0, st>>>(
        row_ptr, col_idx, b->own_first, b->own_count, b->g_own_idx, d_val, s_val, ne, q_mol);
    return cudaGetLastError();
  }
  k_trace<<<(b->count + TR_WARPS - 1) / TR_WARPS, TR_WARPS * 32, 0, st>>>(
      row_ptr, col_idx, b->mol_begin, b->count, nullptr, d_val, s_val, ne, q_mol);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Energy-weighted density and electronic energy.
//   T_j(W) = T_j(D) T_j(H0) T_j(D)   (Eq. 8, 13 PAPER.md:127-129,163-168); only the own columns are kept
//   (PAPER.md:168), and with T_j(D) = 1/2 (I - X) S^-1 they need no n^3 product:
//       y1 = D[:, own]           = 1/2 (t - X t),  t = S^-1[:, own]
//       y2 = H0 y1,   y3 = S^-1 y2,
//       W[:, own] = D (H0 D[:, own]) = 1/2 (y3 - X y3)
//   four n x n x 6 products per submatrix, FP32, bound by reading the dense matrices once each.
// k_thin: out = beta * add + alpha * A * in for one submatrix per blockIdx.y; `in` (n x 6) is staged in
// shared memory, one thread per row, A read column by column (coalesced).  Thin operands live in a
// scratch [submatrix][6][ld]; in_cols / out_blocks switch the first input to columns own0.. of a dense
// matrix and the last output to the column-owned block store.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(DN_THREADS)
k_thin(const int32_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx, int mol_begin, int ld,
       int64_t slab, const float *__restrict__ a, const float *__restrict__ in_thin,
       const float *__restrict__ in_cols, const float *__restrict__ add_thin, float alpha, float beta,
       float *__restrict__ out_thin, float *__restrict__ out_blocks) {
  extern __shared__ float s_in[];  // [6][n]
  const int mat = blockIdx.y;
  const int j = mol_begin + mat;
  const int lo = row_ptr[j];
  const int m = row_ptr[j + 1] - lo;
  const int n = m * NOLSM_BS;
  int l = 0, r_ = m;
  while (l < r_) {
    const int mid = (l + r_) >> 1;
    if (col_idx[lo + mid] < j) l = mid + 1; else r_ = mid;
  }
  const int own0 = l * NOLSM_BS;
  const float *aj = a + (int64_t)mat * slab;
  const int64_t thin0 = (int64_t)mat * NOLSM_BS * ld;
  for (int t = threadIdx.x; t < NOLSM_BS * n; t += blockDim.x) {
    const int p = t / n, k = t - p * n;
    s_in[t] = in_cols ? in_cols[(int64_t)mat * slab + (int64_t)(own0 + p) * ld + k] : in_thin[thin0 + (int64_t)p * ld + k];
  }
  __syncthreads();
  const int r = blockIdx.x * DN_THREADS + threadIdx.x;
  if (r >= n) return;
  float acc[NOLSM_BS];
#pragma unroll
  for (int p = 0; p < NOLSM_BS; ++p) acc[p] = 0.f;
  for (int k = 0; k < n; ++k) {
    const float av = aj[(int64_t)k * ld + r];
#pragma unroll
    for (int p = 0; p < NOLSM_BS; ++p) acc[p] = fmaf(av, s_in[p * n + k], acc[p]);
  }
#pragma unroll
  for (int p = 0; p < NOLSM_BS; ++p) {
    float v = alpha * acc[p];
    if (beta != 0.f) v = fmaf(beta, add_thin ? add_thin[thin0 + (int64_t)p * ld + r] : s_in[p * n + r], v);
    if (out_blocks) out_blocks[(int64_t)lo * 36 + (int64_t)r * NOLSM_BS + p] = v;
    else out_thin[thin0 + (int64_t)p * ld + r] = v;
  }
}

static cudaError_t thin_launch(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx, const float *a,
                               const float *in_thin, const float *in_cols, const float *add_thin, float alpha,
                               float beta, float *out_thin, float *out_blocks, cudaStream_t st) {
  const size_t smem = (size_t)NOLSM_BS * b->max_n * sizeof(float);
  if (smem > 200 * 1024) return cudaErrorInvalidValue;
  if (smem > 48 * 1024) {   // per device: set on every such launch
    cudaError_t e = cudaFuncSetAttribute(k_thin, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  dim3 grid((b->max_n + DN_THREADS - 1) / DN_THREADS, b->count);
  k_thin<<<grid, DN_THREADS, smem, st>>>(row_ptr, col_idx, b->mol_begin, b->ld, (int64_t)b->ld * b->ld, a, in_thin,
                                         in_cols, add_thin, alpha, beta, out_thin, out_blocks);
  return cudaGetLastError();
}

// thin: scratch of 2 * count * 6 * ld floats.  beta with add_thin == nullptr adds beta * (the staged input).
cudaError_t launch_energy_weighted(const nolsm_batch *b, const float *x, const float *sinv, const float *h,
                                   const int32_t *row_ptr, const int32_t *col_idx, float *thin, float *w_val,
                                   cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  float *t0 = thin, *t1 = thin + (size_t)b->count * NOLSM_BS * b->ld;
  cudaError_t e;
  // y1 = 1/2 t - 1/2 X t,  t = S^-1[:, own]
  if ((e = thin_launch(b, row_ptr, col_idx, x, nullptr, sinv, nullptr, -0.5f, 0.5f, t0, nullptr, st)) != cudaSuccess) return e;
  // y2 = H0 y1
  if ((e = thin_launch(b, row_ptr, col_idx, h, t0, nullptr, nullptr, 1.f, 0.f, t1, nullptr, st)) != cudaSuccess) return e;
  // y3 = S^-1 y2
  if ((e = thin_launch(b, row_ptr, col_idx, sinv, t1, nullptr, nullptr, 1.f, 0.f, t0, nullptr, st)) != cudaSuccess) return e;
  // W[:, own] = 1/2 y3 - 1/2 X y3 -> block store
  return thin_launch(b, row_ptr, col_idx, x, t0, nullptr, nullptr, -0.5f, 0.5f, nullptr, w_val, st);
}

// E = sum over the batch's molecules j and their stored blocks k of sum_{o,p} D_k[o][p] H_k[p][o]
// (Eq. 11: D_k = D(i, j) column-owned, H_k = H0(j, i), i = col_idx[k]).  One warp per
// molecule, FP32 products, FP64 accumulation.
__global__ void __launch_bounds__(TR_WARPS * 32)
k_energy(const int32_t *__restrict__ row_ptr, int mol_begin, int count, const float *__restrict__ d_val,
         const float *__restrict__ h_val, double *__restrict__ e_out) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int mat = blockIdx.x * TR_WARPS + warp;
  if (mat >= count) return;
  const int j = mol_begin + mat;
  double sum = 0.0;
  for (int k = row_ptr[j] + lane; k < row_ptr[j + 1]; k += 32) {
    const float *db = d_val + (int64_t)k * 36, *hb = h_val + (int64_t)k * 36;
    double part = 0.0;
#pragma unroll
    for (int o = 0; o < NOLSM_BS; ++o)
#pragma unroll
      for (int p = 0; p < NOLSM_BS; ++p) part += (double)(db[o * NOLSM_BS + p] * hb[p * NOLSM_BS + o]);
    sum += part;
  }
  for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
  if (lane == 0) atomicAdd(e_out, sum);
}

cudaError_t launch_energy(const nolsm_batch *b, const int32_t *row_ptr, const float *d_val, const float *h_val,
                          double *e_out, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  k_energy<<<(b->count + TR_WARPS - 1) / TR_WARPS, TR_WARPS * 32, 0, st>>>(row_ptr, b->mol_begin, b->count, d_val,
                                                                          h_val, e_out);
  return cudaGetLastError();
}
