// Internal declarations shared by the translation units of libnolsm (not part of the C ABI).
// Storage convention for every dense submatrix buffer: COLUMN-major with leading dimension ld
// (element (r,c) at c*ld + r), one slab of ld*ld elements per submatrix, slabs of one logical buffer
// contiguous over the batch.  Column-major is what the tcgen05 epilogue writes coalesced (TMEM lane
// = row), and it makes the A operand M-major and the B operand K-major.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cuda.h>
#include <stdint.h>
#include <string>
#include <vector>
#include "../../include/nolsm.h"

#define NOLSM_BS 6
#define NOLSM_TILE_M 128          // rows per output tile (UMMA M, one CTA)
#define NOLSM_PAD 128             // leading dimensions are multiples of this
#define NOLSM_MAX_RESID_SLOTS 64  // residual history kept per submatrix
#define NOLSM_MAX_HALF 14         // FP16 operand buffers of a batch (6 / 10 of the iterations in FP16 / FP32 mode
                                  // + 4 of a gathered batch: split copies of S and H written by the builder)
#define NOLSM_MAX_UNIT 11         // FP32 buffers of a batch (the FP16 buffers alias units 4..)

struct TileDesc {                 // one output tile of one submatrix
  int32_t mat;                    // index inside the batch
  int32_t m0, n0;                 // first row / column
  int32_t nt;                     // columns in this tile (multiple of 64, <= BN)
};

enum { EPI_AXPBY = 0, EPI_IDENT = 1 };

// Parameters of one batched product  C = epilogue(A * B)  over a tile list.
struct GemmParams {
  const TileDesc *tiles;
  int32_t n_tiles;
  const int32_t *dims;            // true dimension n_j per submatrix
  const int32_t *state;           // per submatrix: last iteration index it executes (may be null)
  int32_t iter;                   // tile runs iff state==null or iter <= state[m]
  int32_t ld;
  int64_t slab;                   // ld*ld
  int32_t mode;                   // EPI_*
  float alpha, beta;
  const float *alpha_div;         // optional per-submatrix divisor of alpha (S^-1 = Z^2 / s_S)
  const float *a32, *b32;         // SIMT operands
  const float *cin32;             // AXPBY input (may alias cout32)
  float *cout32;                  // FP32 output (may be null in IDENT mode of the FP16 path)
  __half *cout16;                 // FP16 copy of the output (tcgen05 path; may be null)
  __half *cout16_lo;              // split path: residual part, scaled by 2^11 (may be null)
  float *resid2;                  // IDENT: per-submatrix sum of squares of the output (atomicAdd)
};

// One product of a chain (chain_umma.cu).  Buffer indices refer to the batch's FP16 buffers h[] and
// FP32 units u[]; entries indexed by the iteration parity implement the ping-pong of the iterates.
struct ChainOp {
  int32_t a[2], b[2];             // FP16 operands (hi parts), by iteration parity
  int32_t a_lo[2], b_lo[2];       // lo parts of split operands (FP32-quality product), -1: plain FP16
                                  // a_lo set, b_lo -1: only the left operand is split (the right one is exact in FP16)
  int32_t out16[2], out16_lo[2];  // FP16 copy of the result (hi [, lo * 2^11]), -1: none
  int32_t cin32, cout32;          // FP32 units read (AXPBY, beta != 0) / written, -1: none
  int32_t cin16[2];               // instead of cin32: the add-in is an FP16 buffer (by parity), -1: none.  For
                                  // iterations whose result is refined afterwards: no FP32 master is kept
  int32_t cin16_lo[2];            // lo part of a split add-in (master iterate kept as hi + lo * 2^-11), -1: none
  int32_t lo_stream;              // 1: out16_lo / cin16_lo are touched once per iteration and never by an MMA: streaming
                                  // (evict-first) loads and stores, so that they do not take L2 from the operands
  int32_t mode;                   // EPI_IDENT: I - A B     EPI_AXPBY: beta * Cin + alpha * A B
  int32_t resid;                  // 1: ||result||_F^2 over the true n x n part drives the stop rule
  int32_t colnorm;                // 1 (with resid, EPI_IDENT): the column sums of |result| are accumulated too, so that
                                  // ||result||_1 is known when the product completes (ChainProgram::tol_pred)
  int32_t use_div;                // 1: alpha /= alpha_div[submatrix]; 2: alpha, beta and diag
  float alpha, beta;
  float diag;                     // AXPBY: + diag * I (after the division)
};

struct ChainProgram {
  ChainOp ops[3];
  int32_t n_ops;                  // products per iteration, strictly ordered per submatrix
  int32_t max_iter, fixed_iter;   // fixed_iter > 0: exactly that many iterations, no residual test
  float tol;                      // stop rule of DESIGN.md reading 9 on the residual of the `resid` op
  int32_t group;                  // window: submatrices in flight together (L2 residency)
  int32_t parity_from_iters;      // 1: the operand tables are indexed by the parity of the LAST full iteration of
                                  // the chain that ran before on this batch ((iters[m] + 1) & 1) instead of the
                                  // own iteration's: lets a one-shot product read the final FP16 iterate in place
  int32_t use_alpha_tab;          // 1: per-submatrix, per-iteration scaling alpha_k from nolsm_batch::d_alpha
  int32_t stop_early;             // 1: the iteration whose residual passes the test is NOT finished (its
                                  // remaining products are skipped); 0: it is (reading 9, "+1 rule")
  float rescale_target;           // ops with colnorm == 2: |eigenvalue| the bound on rho(X0) is mapped to (and cap of the factor)
  int32_t skip_tail;              // ops at the end of an iteration that the LAST iteration of a chain without stop_early
                                  // does not need (Eq. 15-17 with ops E, Z, Y: 1 -- nothing reads the final Y)
  float tol_pred;                 // > 0 (with stop_early, Eq. 15-17 only, ops ordered E, Z, Y): a-priori stop.  With
                                  // E_k = I - Z_k Y_k symmetric, E_{k+1} = 3/4 E_k^2 + 1/4 E_k^3 exactly, hence
                                  // ||E_{k+1}||_2 <= 3/4 b^2 + 1/4 b^3 with b = ||E_k||_1 >= ||E_k||_2.  When that bound
                                  // is <= tol_pred, iteration k only runs its Z update (op 1) and the submatrix is
                                  // done: Y_{k+1} and the product E_{k+1} that would only confirm it are never formed
};

// nolsm_batch::d_colpart holds colpart_strips(ld) * count * ld floats: the column partial sums of the norm bounds
// (one strip per 128 rows) and, during a chain launch with an a-priori stop, four iteration slots of column sums
// plus one strip of maxima (chain_engine.cu)
inline int colpart_strips(int ld) { return std::max((ld + 127) / 128, 5); }

struct nolsm_batch {
  int32_t count = 0, ld = 0, mol_begin = 0, max_n = 0, slot = 0;
  float inv_scale = 0.5f;         // s_S = inv_scale * max(1, bound)   (reading 7; 1 with NOLSM_FLAG_UNIT_SCALE)
  float sign_scale = 1.f / 1.5f;  // s_j = sign_scale * bound          (reading 5; 1 with NOLSM_FLAG_UNIT_SCALE)
  bool x_pending = false;         // the sign chain stopped after E_k = I - X_k^2 passed the test: the update
                                  // X_{k+1} = X_k + 1/2 X_k E_k is folded into the density columns (reading 9)
  bool x_pending_split = false;   // E_k is stored as hi + lo (FP32 mode)
  const int32_t *row_ptr = nullptr, *col_idx = nullptr;   // pattern the batch was built from (caller-owned, sparse batches)
  // combined submatrices (nolsm_build_submatrices_grouped): submatrix m of the batch is group mol_begin + m
  bool grouped = false;
  const int32_t *g_own_ptr = nullptr, *g_own_idx = nullptr, *g_list_ptr = nullptr, *g_list_idx = nullptr;
  int32_t own_first = 0, own_count = 0;   // the batch's owners: g_own_idx[own_first, own_first + own_count)
  int32_t sinv_hi = -1, sinv_lo = -1;   // >= 0: S^-1 lives as the split pair h[sinv_hi] + h[sinv_lo] * 2^-11 and u[2] holds
  bool sinv32_full = true;              // only its own columns in FP32 until join_sinv (false)
  bool x0_built = false;                // X0 for mu = x0_mu is in place (written by the prepare stage), d_scale set
  double x0_mu = 0.0;
  bool b32_built = true;                // u3 holds B (false: the whole path went from B0 straight to X0)
  bool lowdin = false;                  // prepared in the symmetric Loewdin form (NOLSM_FLAG_LOWDIN): u3 = S^-1/2 H S^-1/2,
                                        // own columns of u2 = (s_S S^-1)^1/2 = Z, Z as split pair in (h6, h7), s_S in d_scale_s
  bool sinv_own_only = false;           // S^-1 was refined in its own columns only (nolsm_solve_mu): no full S^-1
  int32_t sign_iter0 = 0;         // iterations of the last sign chain that ran before its adaptive launch (0 or 1: the rescaled
                                  // first iteration has a launch of its own); d_iters counts from there
  int32_t sign_ops = 2;           // products per sign iteration of the last chain (3 with NOLSM_FLAG_ORDER3)
  bool x_split = false;           // the sign iterate lives as hi (h[iters & 1]) + lo * 2^-11 (h[2]); u[0] holds X in
  bool x32_valid = false;         // FP32 only after join_x (reading 12)
  bool s_split_built = false;     // the builder wrote the split copy of S into h[n_half-4], h[n_half-3]
  bool s32_built = true;          // u0 holds the FP32 T_j(S) (false: nolsm_solve_mu built the split copy only)
  bool s_norm_built = false;      // d_norm_s holds ||S_j||_1 = ||S_j||_inf from the builder
  bool prefer_pair = false;       // batch shape favours the pair engine (nolsm.h, NOLSM_FLAG_*)
  bool engine_simt = false;       // prepared by the FP32 SIMT debugging path (different buffer roles)
  bool sparse = true;             // false: dense microbench batch (no neighbour list)
  bool prepared = false;          // S^-1 and B available
  int32_t prepared_precision = -1;
  int32_t x_parity = 0;           // FP32 mode: which ping-pong buffer holds X per submatrix -> d_iters parity
  std::vector<int32_t> n_host;
  // device
  void *base = nullptr;           // dense workspace of this slot
  size_t base_bytes = 0;
  int32_t *d_dims = nullptr;      // [count]
  int32_t *d_state = nullptr;     // [count]
  int32_t *d_iters = nullptr;     // [count]
  float *d_resid2 = nullptr;      // [NOLSM_MAX_RESID_SLOTS][count]
  float *d_lastres = nullptr;     // [count]
  float *d_scale = nullptr;       // [count] s_j of the sign scaling
  float *d_alpha = nullptr;       // [count][8] alpha_k of the scaled Newton-Schulz start (gap_hint)
  float *d_norm = nullptr;        // [2][count] scratch for norm bounds
  float *d_scale_s = nullptr;     // [count] s_S of the Loewdin form (d_scale is reused by the sign iteration)
  float *d_norm_s = nullptr;      // [2][count] norm bound of S from the builder (s_norm_built)
  float *d_colpart = nullptr;     // [count][ld/128][ld] column-sum shares of the row strips (k_norm_bound)
  size_t colpart_cap = 0;
  int32_t *d_active = nullptr;    // [NOLSM_MAX_RESID_SLOTS] active counters per iteration
  TileDesc *d_tiles_simt = nullptr; // 128x128 tiles for the SIMT kernel
  int32_t n_tiles_simt = 0;
  size_t meta_cap = 0;            // capacity (in submatrices) of the metadata arrays
  size_t tiles_simt_cap = 0;
  double sum_n3 = 0.0, sum_n3_padded = 0.0;
  // logical buffers (set by layout_batch): fp32 units u[0..6], fp16 halves h[0..5] alias units 4..6
  float *u[NOLSM_MAX_UNIT] = {nullptr};
  __half *h[NOLSM_MAX_HALF] = {nullptr};
  int32_t n_half = 6, n_unit = 7; // buffers laid out in this batch (precision dependent)
  unsigned long long *d_slot_state = nullptr;      // [count] chain engine: window slots (chain_epilogue.cuh)
  int32_t *d_slot_done = nullptr; // [count] chain engine: completed tiles of a slot's current op
  int32_t *d_sched = nullptr;     // [4] chain engine: next submatrix to admit, retired slots, unconverged count
  unsigned long long *d_tile_counter = nullptr;   // chain engine: next tile index to claim
  float *d_thin = nullptr;        // [2][count][6][ld] scratch of the thin products (energy-weighted density)
  size_t thin_cap = 0;            // floats
  CUtensorMap *d_maps = nullptr;  // device array: n_half FP16 maps {64,64,1}, then n_unit FP32 maps {32,32,1}
  bool maps_valid = false;
};

struct nolsm_ctx {
  nolsm_config cfg;
  bool inv_refine_default = true;   // the caller left nolsm_config.inv_refine < 0
  int device = 0;
  int sm_count = 148;
  size_t l2_bytes = 0;
  std::string err;
  std::vector<nolsm_batch *> slots;
  int64_t launches = 0;
  double *d_scalars = nullptr;    // [4] device doubles: ne, ne_diag, spare
  double *h_scalars = nullptr;    // pinned mirror
  int32_t *h_active = nullptr;    // pinned [NOLSM_MAX_RESID_SLOTS]
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  cudaEvent_t tev[2] = {nullptr, nullptr};   // timing of the sign-iteration chain kernel
  void *encode_tiled = nullptr;   // cuTensorMapEncodeTiled entry point
  bool eval_energy = false;       // nolsm_evaluate in progress: also E (and W) per batch
  nolsm_bsr *eval_w = nullptr;
  bool umma_ok = false;
  bool pair_ok = false;           // pair-CTA (cta_group::2) engine usable
  int pair_clusters = 0;          // co-resident CTA pairs
  // device mirrors of the caller's HOST store (nolsm_solve_mu_host), grown on demand
  int32_t *m_row_ptr = nullptr, *m_col_idx = nullptr;
  float *m_h = nullptr, *m_s = nullptr, *m_d = nullptr;
  size_t m_cap_mol = 0, m_cap_nnzb = 0;
  bool has_model = false;         // nolsm_set_model: builds evaluate the model instead of gathering
  nolsm_model model;
};

#define NOLSM_CUDA(ctx, call)                                                          \
  do {                                                                                 \
    cudaError_t e__ = (call);                                                          \
    if (e__ != cudaSuccess) {                                                          \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);                \
      return NOLSM_ECUDA;                                                              \
    }                                                                                  \
  } while (0)

static inline int32_t round_up(int32_t x, int32_t g) { return (x + g - 1) / g * g; }

// ---- launchers implemented in the kernel translation units (all asynchronous on `st`) ----
// sparse side
cudaError_t launch_neighbour_count(int n_mol, const int32_t *pos, const int32_t *box, int32_t rc,
                                   int32_t *counts, cudaStream_t st);
cudaError_t launch_exclusive_scan(const int32_t *counts, int32_t *row_ptr, int n, cudaStream_t st);
cudaError_t launch_neighbour_fill(int n_mol, const int32_t *pos, const int32_t *box, int32_t rc,
                                  const int32_t *row_ptr, int32_t *col_idx, cudaStream_t st);
cudaError_t launch_generate(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx,
                            const nolsm_model *model, float *h_out, float *s_out, bool split_s,
                            cudaStream_t st);
cudaError_t launch_gather(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx,
                          const int32_t *list_ptr, const int32_t *list_idx,
                          const float *h_val, const float *s_val, float *h_out, float *s_out, bool split_s,
                          float *s_norm, cudaStream_t st);

// own columns of S^-1 (u2) to / from a packed [count][6][ld] array (operator cache of nolsm_solve_mu)
cudaError_t launch_pack_square(const nolsm_batch *b, float *dense, float *packed, bool save, cudaStream_t st);
cudaError_t launch_own_columns(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx, float *mat,
                               float *packed, bool save, cudaStream_t st);
// the sign iterate as the kernels of a5 read it: FP32, or split hi (by the parity of iters) + lo
struct XRef {
  const float *x32;
  const __half *hi0, *hi1, *lo0, *lo1;   // hi0 != null: split pair (hi, lo) number (iters & 1)
};
cudaError_t launch_join_split(const nolsm_batch *b, const XRef &x, float *dst32, cudaStream_t st);
cudaError_t launch_expand_store(int n_mol, const int32_t *rp_src, const int32_t *ci_src, const float *val_src,
                                const int32_t *rp_dst, const int32_t *ci_dst, float *val_dst, cudaStream_t st);
cudaError_t launch_own_join_grouped(const nolsm_batch *b, const __half *hi, const __half *lo, float *dst32,
                                    cudaStream_t st);
cudaError_t launch_density_grouped(const nolsm_batch *b, const XRef &x, const float *sinv, const int32_t *row_ptr,
                                   const int32_t *col_idx, float *d_val, cudaStream_t st);
// own columns of a split matrix (hi + lo * 2^-11) as FP32 into the same columns of dst32
// thin_kernels.cu
cudaError_t launch_density_split(const nolsm_batch *b, const XRef &x, const float *sinv, const int32_t *row_ptr,
                                 const int32_t *col_idx, float *d_val, double *ne_diag, const __half *e_hi,
                                 const __half *e_lo, float *u_thin, cudaStream_t st, float *thin_out = nullptr);
cudaError_t launch_scaled_out(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx, const __half *a_hi,
                              const __half *a_lo, float *thin_in, const float *scale, float *d_val, cudaStream_t st);
cudaError_t launch_own_refine(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx, const __half *s_hi,
                              const __half *s_lo, const __half *a0, float *thin, float *out32, int rounds,
                              cudaStream_t st);
cudaError_t launch_own_join(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx, const __half *hi,
                            const __half *lo, float *dst32, cudaStream_t st);
cudaError_t launch_density(const nolsm_batch *b, const XRef &x, const float *sinv,
                           const int32_t *row_ptr, const int32_t *col_idx, float *d_val,
                           double *ne_diag, const __half *e_hi, const __half *e_lo, float *u_thin,
                           cudaStream_t st);
cudaError_t launch_trace(const nolsm_batch *b, const int32_t *row_ptr, const int32_t *col_idx,
                         const float *d_val, const float *s_val, double *ne, double *q_mol,
                         cudaStream_t st);
cudaError_t launch_energy_weighted(const nolsm_batch *b, const float *x, const float *sinv, const float *h,
                                   const int32_t *row_ptr, const int32_t *col_idx, float *thin, float *w_val,
                                   cudaStream_t st);
cudaError_t launch_energy(const nolsm_batch *b, const int32_t *row_ptr, const float *d_val, const float *h_val,
                          double *e_out, cudaStream_t st);
// dense helpers
cudaError_t launch_norm_bound(const nolsm_batch *b, const float *a, float mu, bool symmetric, float *norm2,
                              cudaStream_t st);
cudaError_t launch_canon_pair(const nolsm_batch *b, const int32_t *iters, const __half *hi0, const __half *lo0,
                              __half *hi1, __half *lo1, cudaStream_t st);
cudaError_t launch_norm_bound16(const nolsm_batch *b, const __half *a, float mu, float *norm2, cudaStream_t st);
cudaError_t launch_x0_scale(const nolsm_batch *b, const float *norm2, float slack, float *scale_out, cudaStream_t st);
cudaError_t launch_init_inverse(const nolsm_batch *b, const float *s, const float *norm2, float *y32,
                                float *z32, __half *y16, __half *z16, __half *y16_lo, __half *z16_lo,
                                float *scale_out, cudaStream_t st);
// lean start of Eq. 15-17 in FP16 mode: only Z1 = 3/2 I - 1/2 S/s_S is formed; Y1 = (S_hi Z1)/s_S is a product
cudaError_t launch_init_z1(const nolsm_batch *b, const __half *s_hi, const __half *s_lo, const float *norm2, __half *z16,
                           float *scale_out, cudaStream_t st);
cudaError_t launch_init_inverse_first(const nolsm_batch *b, const float *s, const float *norm2, float *y32,
                                      float *z32, __half *y16, __half *y16_lo, __half *z16, __half *z16_lo,
                                      __half *e16, __half *e16_lo, float *scale_out, cudaStream_t st);
// alpha_k schedule of the scaled start from the scale s_j (d_scale) and a lower bound `gap` on |lambda - mu|
cudaError_t launch_alpha_schedule(const nolsm_batch *b, const float *scale, float gap, float *alpha_tab,
                                  cudaStream_t st);
cudaError_t launch_make_x0(const nolsm_batch *b, const float *bmat, float mu, const float *norm2,
                           const float *scale_in, float *x32, __half *x16, __half *x16_lo, float *scale_out,
                           cudaStream_t st);
cudaError_t launch_scale_copy(const nolsm_batch *b, const float *src, const float *scale, int invert,
                              float *dst32, __half *dst16, __half *dst16_lo, cudaStream_t st);
cudaError_t launch_control(const nolsm_batch *b, int phase, int iter, float tol, int max_iter,
                           int fixed_iter, cudaStream_t st);
cudaError_t launch_pack(const float *src_rowmajor, int n, int batch, int ld, float *dst, int pad_identity,
                        cudaStream_t st);
cudaError_t launch_unpack(const float *src, int ld, int64_t slab, const int32_t *iters_parity,
                          const float *src_alt, int n, int batch, float *dst_rowmajor, cudaStream_t st);
cudaError_t launch_gemm_simt(const GemmParams &p, cudaStream_t st);
// tcgen05 path
nolsm_status umma_init(nolsm_ctx *ctx);
nolsm_status umma_make_maps(nolsm_ctx *ctx, nolsm_batch *b);
cudaError_t launch_chain(nolsm_ctx *ctx, const nolsm_batch *b, const ChainProgram &prog, const float *alpha_div,
                         bool touch_stats, cudaStream_t st);
