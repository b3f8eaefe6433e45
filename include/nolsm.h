/* nolsm.h -- C ABI of the B200-native NOLSM hot path (arXiv 2104.08245).
 *
 * The path (PAPER.md = the paper text; DESIGN.md lists every reading taken):
 *   a0  neighbour lists / index sets            Fig. 2 b,c  PAPER.md:172,190; merged pattern :158
 *   a1  dense submatrices T_j(H), T_j(S)        step (i)    PAPER.md:140; NOLSM :158
 *   a1' the same from positions + a model     Fig. 2 d,e  PAPER.md:172,202 (nolsm_set_model)
 *   a2  S_j^-1 by the coupled Newton-Schulz     Eq. 15-17
 *   a3  B_j = S_j^-1 H_j, X0 = (B_j - mu I)/s   Eq. 12      PAPER.md:160; rescaling :138
 *   a4  sign iteration X <- 1/2 X (3I - X^2)    Eq. 9-10
 *   a5  D_j[:,own] = 1/2 (I - X) S_j^-1[:,own]  Eq. 12
 *   a6  write-back of the own columns           step (iii)  PAPER.md:142; Fig. 2 h,i :172-178
 *   a7  N(mu) = 2 tr(DS), bisection on mu
 *
 * Conventions
 *   - Every array pointer is a DEVICE pointer unless the parameter comment says "host".  The caller
 *     allocates and owns every array it passes; the context owns only scratch (workspaces, tensor
 *     maps, statistics).  `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - Calls are asynchronous on `stream` except where a scalar must reach the host; those calls
 *     say "synchronises".
 *   - Errors are return codes; nothing throws across this boundary.  nolsm_last_error() gives text.
 *   - Block-sparse matrices are CSR of uniform bs x bs blocks (bs = 6), FP32, block row-major.
 *     H and S: block k of row i is block (i, col_idx[k]).  D is column-owned: block k
 *     of row j holds D(col_idx[k], j), i.e. the rows of neighbour col_idx[k] in the own columns of
 *     the submatrix of molecule j.  H, S and D share one pattern (row_ptr/col_idx = neighbour list,
 *     ascending within a row, self included).
 *   - There is no CPU fallback.  Without a CUDA device every compute entry returns NOLSM_ECUDA.
 */
#ifndef NOLSM_H
#define NOLSM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* exported symbols: the library is built with -fvisibility=hidden and exports only these entry points */
#if defined(__GNUC__)
#define NOLSM_API __attribute__((visibility("default")))
#else
#define NOLSM_API
#endif

typedef struct nolsm_ctx nolsm_ctx;     /* opaque: workspaces, tensor maps, statistics */
typedef struct nolsm_batch nolsm_batch; /* opaque, owned by the context: one batch of dense submatrices */

typedef enum {
  NOLSM_OK = 0,
  NOLSM_EINVAL = 1,   /* bad argument (null pointer, negative size, unsupported block size, ...) */
  NOLSM_ENOMEM = 2,   /* device or host allocation failed / workspace too small for one submatrix */
  NOLSM_ECUDA = 3,    /* a CUDA call failed (no device, launch error); see nolsm_last_error */
  NOLSM_ENOTSPD = 4,  /* Eq. 15-17 ended at inv_max_iter or on a NaN for at least one submatrix: S_j not SPD / badly
                         scaled (PAPER.md:203-215 needs ||I - Y_0|| < 1).  Counted on the device: returned by
                         nolsm_sign_batched and the whole-path calls with or without a stats struct */
  NOLSM_ENOCONV = 5,  /* the sign iteration ended at max_iter or on a NaN for at least one submatrix (whole-path
                         calls: on the FINAL mu; intermediate bisection steps may sit inside a band).  Counted on
                         the device, independent of stats.  The outputs are written all the same */
  NOLSM_EBRACKET = 6  /* nolsm_solve_mu with tol_ne_per_mol >= 0: the bisection ended outside the tolerance without
                         ever moving one end of [mu_lo, mu_hi]: N(mu) - N_e kept one sign at every midpoint */
} nolsm_status;

typedef enum {
  NOLSM_FP16_FP32 = 0, /* FP16 operands, FP32 accumulate, FP32 master iterates */
  NOLSM_FP32 = 1       /* FP32-quality products everywhere */
} nolsm_precision;

typedef struct {
  int32_t precision;        /* nolsm_precision */
  float tol;                /* sign-iteration stop: r_k = ||X_k^2 - I||_F / sqrt(n) < tol, then ONE more
                               iteration is finished (reading 9).  <= 0: 1e-2 (FP16) / 1e-5 (FP32) */
  int32_t max_iter;         /* cap on sign iterations (default 30 if <= 0) */
  int32_t fixed_iter;       /* > 0: run exactly this many sign iterations, no residual test */
  float inv_tol;            /* stop of Eq. 15-17 on r_k = ||I - Z_k Y_k||_F / sqrt(n) < inv_tol.  Without a
                               refinement behind it iteration k is finished first (as for the sign iteration);
                               with one (inv_refine > 0) Z_k is taken as it is and the two products that would
                               finish iteration k are skipped.  <= 0: 3e-3 (FP16 with refinement), 1e-2 (FP16
                               without), 1e-5 (FP32) */
  int32_t inv_max_iter;     /* cap on Eq. 15-17 iterations (default 20 if <= 0) */
  int32_t inv_refine;       /* FP32-quality Newton refinements of S^-1 after Eq. 15-17 (reading 11);
                               < 0: default 1;  0 in FP16 mode = the paper-literal all-FP16 S^-1 */
  int64_t workspace_bytes;  /* upper bound on the dense workspace the context may allocate (<= 0: 24 GiB) */
  int32_t group;            /* window: submatrices in flight together inside one iteration kernel; a submatrix that
                               converges hands its place to the next one of the batch (<= 0: chosen by the context
                               from the L2 size and the tile count) */
  int32_t flags;            /* NOLSM_FLAG_* */
  float gap_hint;           /* > 0: a lower bound on |lambda - mu| over the spectra of the S_j^-1 H_j (e.g. half the
                               HOMO-LUMO gap of the previous MD step).  The sign iteration then starts with scaled
                               steps X <- 1/2 a_k X (3I - a_k^2 X^2), a_k = sqrt(3/(1 + l_k + l_k^2)), l_0 = gap_hint/s_j
                               (DESIGN.md section 8), which saves iterations; a bound that is wrong
                               costs iterations, never convergence.  0: the plain iteration of Eq. 9 (default). */
  int64_t cache_bytes;      /* nolsm_solve_mu with several mu steps, batches streamed through the workspace:
                               upper bound on the device memory used to keep B_j and the own columns of S_j^-1
                               of every submatrix from the first step, so that later steps skip a1-a3 (gather,
                               Eq. 15-17, refinement, B = S^-1 H).  0: what is free at the call, less
                               workspace_bytes and 4 GiB;  < 0: off.  4 (n_j^2 + 6 ld) bytes per submatrix; when
                               that does not fit, the steps recompute.  Freed before the call returns. */
} nolsm_config;

/* Engine of the matrix iterations.  With neither PAIR nor SINGLE set the context picks per batch:
 * the pair engine when its 256-row tiles waste little (sum of the dimensions padded to 256 at most 4 % above
 * the sum padded to 128) and the mean dimension is at least 1100 -- where it measured 5-11 % ahead -- else
 * the single-CTA engine.  Each engine is bitwise reproducible run to run; different engines round differently. */
#define NOLSM_FLAG_SIMT_ONLY 1 /* debugging: run every product on the FP32 SIMT kernel */
#define NOLSM_FLAG_PAIR 2      /* always the CTA-pair engine (tcgen05 cta_group::2, 256-row tiles) */
#define NOLSM_FLAG_SINGLE 8    /* always the single-CTA engine (128-row tiles) */
#define NOLSM_FLAG_ORDER3 32    /* SURVEY 8(f)#4, "higher-order Pade approximants / arbitrary-order schemes": the
                                  third-order member X <- X (I + 1/2 E + 3/8 E^2), E = I - X^2 (three products per
                                  iteration, residual E -> 5/8 E^3) instead of Eq. 9's second-order one.  FP16/FP32 mode
                                  only; the last iteration is then not folded into the density columns */
#define NOLSM_FLAG_NO_PREDICT 64 /* Eq. 15-17, FP16 mode: do not use the a-priori stop (reading 11: from
                                  ||E_k||_1 the bound 3/4 b^2 + 1/4 b^3 >= ||E_{k+1}||_2 is known before iteration k
                                  is finished; when it is small enough only Z_{k+1} is formed).  With this flag every
                                  stop is decided on a measured residual: two products more per submatrix, same iterate.
                                  In FP32 mode nolsm_solve_mu then iterates Eq. 15-17 on split operands to inv_tol
                                  instead of refining twice */
#define NOLSM_FLAG_LOWDIN 128    /* SURVEY 8(f)#4, symmetric Loewdin form (nolsm_solve_mu, FP32 mode only): with Z = (S_j/s)^-1/2
                                  from Eq. 15-17 run to its end on split operands, the sign function is taken of the
                                  SYMMETRIC A~ = Z H_j Z / s - mu I = S^-1/2 H S^-1/2 - mu I, and
                                  D_j[:, own] = Z (1/2 (I - sign A~)) Z[:, own] / s.  Same D as the non-orthogonal
                                  form of Eq. 12 up to rounding; no S^-1, no B */
#define NOLSM_FLAG_NO_RESCALE 256 /* do not rescale the first sign iteration.  By default the first product of
                                  the iteration (X0^2) also yields ||X0^2||_1 >= rho(X0)^2, a tighter bound on the
                                  spectrum than the O(n^2) norm bound X0 was scaled with, and iteration 0 is applied to
                                  a X0, a = 1.7 / sqrt(||X0^2||_1) >= 1 ("rescaled so that its spectrum
                                  lies in the convergence region"; reading 5): one iteration fewer on the
                                  water systems, same sign function */
#define NOLSM_FLAG_UNIT_SCALE 16 /* scale by the norm bound itself: Y0 = S/bound, X0 = A/bound (spectra in (0,1] and
                                  [-1,1]) instead of bound/2 and bound/1.5 (readings 5, 7); costs one
                                  iteration each */

typedef struct {            /* CSR of uniform bs x bs FP32 blocks; all pointers device, caller-owned */
  int32_t n_mol;            /* block rows = molecules */
  int32_t bs;               /* block size, must be 6 */
  const int32_t *row_ptr;   /* [n_mol+1] */
  const int32_t *col_idx;   /* [nnzb], ascending within a row */
  float *val;               /* [nnzb*bs*bs], each block row-major; 16-byte aligned */
} nolsm_bsr;

typedef struct {            /* filled by nolsm_sign_batched (host struct) */
  int32_t n_sub;            /* submatrices in the batch */
  int32_t iter_min, iter_max;   /* sign iterations executed per submatrix */
  int64_t iter_sum;
  int32_t n_unconverged;    /* submatrices that hit max_iter with r >= tol */
  float worst_residual;     /* max over submatrices of the last residual r_k that was measured */
  int64_t gemms;            /* n x n x n products executed by this call (all kinds) */
  double flops_sign;        /* 2 n^3 per executed sign-iteration GEMM, n = TRUE dimension */
  double flops_sign_padded; /* same with the padded tile extents */
  double flops_prepare;     /* Eq. 15-17, refinement and B = S^-1 H, if this call ran them */
  int32_t inv_iter_max;     /* Eq. 15-17 iterations executed (0 if the batch was already prepared) */
  float inv_worst_residual;
  float ms_chain;           /* CUDA-event time of the sign-iteration kernel alone (all iterations of the batch) */
  float chain_mcycles;      /* SM cycles of that kernel (max over its CTAs), in millions: ms_chain and this give the
                               SM clock the kernel ran at under the power cap */
} nolsm_sign_stats;

typedef struct {            /* filled by nolsm_solve_mu (host struct) */
  int32_t mu_steps;         /* N(mu) evaluations performed */
  int32_t n_batches;
  int32_t resident;         /* 1 if every batch stayed in the workspace across mu steps (S^-1, B reused) */
  int32_t cached;           /* 1 if B_j and S_j^-1[:,own] were kept in the operator cache instead (cache_bytes) */
  double mu_lo, mu_hi;      /* final bracket */
  double ne_diag;           /* cross-check: sum_j sum_{c in own_j} (1 - X_cc) of the last step (reading 15) */
  nolsm_sign_stats last;    /* statistics of the last mu step, summed over batches */
  double flops_sign_total;  /* over all mu steps */
  double flops_prepare_total;
  float ms_gather, ms_prepare, ms_sign, ms_density; /* CUDA-event times summed over batches and steps */
  float ms_chain;           /* of ms_sign: the sign-iteration kernel alone (without norm bound and X0) */
  int32_t chain_launches;   /* launches of that kernel behind ms_chain */
} nolsm_solve_stats;

/* Context.  `cfg` may be NULL (defaults).  Returns NOLSM_ECUDA when no device is usable. */
NOLSM_API nolsm_status nolsm_create(nolsm_ctx **ctx, const nolsm_config *cfg);
NOLSM_API void nolsm_destroy(nolsm_ctx *ctx);
NOLSM_API const char *nolsm_last_error(const nolsm_ctx *ctx); /* ctx may be NULL: last error of nolsm_create */
NOLSM_API int32_t nolsm_version(void);

/* a0: neighbour list of every molecule from integer positions.
 * pos_q [n_mol*3] int32 grid units in [0, box_q); box_q host int32[3], each even; rc_q cutoff in grid
 * units.  Pair (i,j) is kept iff the per-axis minimum-image distance satisfies dx^2+dy^2+dz^2 <= rc_q^2
 * in int64 (closed ball, self included).  Output CSR: row_ptr [n_mol+1], col_idx ascending per row.
 * Two passes inside; if the list needs more than `cap` entries nothing is written to col_idx and
 * NOLSM_ENOMEM is returned with *nnzb_out set to the needed size.  Synchronises (nnzb reaches the host). */
NOLSM_API nolsm_status nolsm_build_neighbours(nolsm_ctx *ctx, int32_t n_mol, const int32_t *pos_q,
                                    const int32_t *box_q /*host*/, int32_t rc_q, int32_t *row_ptr,
                                    int32_t *col_idx, int64_t cap, int64_t *nnzb_out /*host*/, void *stream);

/* a0 without device-memory allocation, for callers that cannot call cudaMalloc (serving loops, harnesses that forbid
 * it).  Same arguments, kernels, result and status codes as nolsm_build_neighbours; the neighbour counts between the
 * two passes live in a static device array of NOLSM_STATIC_MAX_MOL int32 (1 MiB per device that loads the library,
 * held until the process exits) instead of a cudaMalloc'ed buffer.  n_mol > NOLSM_STATIC_MAX_MOL returns NOLSM_EINVAL
 * (text in nolsm_last_error).  No cudaMalloc / cudaFree / allocating library call is made.  ctx may be NULL (then no
 * error text and no launch count are kept).  Every call on a device shares the array: calls that overlap on the GPU
 * (different streams or threads) race -- serialise them; nothing in it needs clearing between calls (every count that
 * is read was written by the same call).  Synchronises the stream like nolsm_build_neighbours (nnzb reaches the host).
 * nolsm_static_setup resolves the array's device address for the CURRENT device (once per device; optional, the first
 * nolsm_build_neighbours_static on a device does it otherwise). */
#define NOLSM_STATIC_MAX_MOL 262144
NOLSM_API nolsm_status nolsm_static_setup(void);
NOLSM_API nolsm_status nolsm_build_neighbours_static(nolsm_ctx *ctx, int32_t n_mol, const int32_t *pos_q,
                                           const int32_t *box_q /*host*/, int32_t rc_q, int32_t *row_ptr,
                                           int32_t *col_idx, int64_t cap, int64_t *nnzb_out /*host*/, void *stream);

/* a1: gather molecules [mol_begin, mol_begin+mol_count) into a context-owned batch
 * of dense submatrix pairs T_j(H), T_j(S): entry ((a,o),(b,p)) = block (N_j[a], N_j[b]) of the store if
 * that pair is stored, else 0.  H and S must share row_ptr/col_idx.  *out stays valid until the next
 * nolsm_build_submatrices on the same slot, nolsm_release_batch or nolsm_destroy; no other entry point touches
 * it (nolsm_solve_mu, nolsm_evaluate, nolsm_solve_mu_host, nolsm_sign_dense_batched and nolsm_gemm_batched work
 * in context-private slots).  `slot` in [0, 4096) selects one of the caller's batch slots (0 for streaming use).
 * The batch keeps H->row_ptr / H->col_idx (not the values): they must stay alive while the batch is used.
 * Synchronises once (reads mol_count+1 row pointers) to size the batch.  NOLSM_ENOMEM if the caller's batches
 * plus this one exceed workspace_bytes. */
NOLSM_API nolsm_status nolsm_build_submatrices(nolsm_ctx *ctx, const nolsm_bsr *H, const nolsm_bsr *S,
                                     int32_t mol_begin, int32_t mol_count, int32_t slot,
                                     nolsm_batch **out, void *stream);
/* a1', SURVEY 8(f)#2 (Fig. 2 d-e: "the matrix elements of the submatrices are
 * generated on the accelerator, only the index metadata crosses"): a two-centre model from which the
 * elements of T_j(H), T_j(S) are evaluated on the device instead of being gathered from the block
 * stores.  Molecule i has n_site = 3 sites at pos_i + site_offset[s]; basis function o sits on site
 * orb_site[o].  For a stored pair (ia, ib) (centre distance <= rc_q, integer minimum image as in
 * nolsm_build_neighbours) and functions o on ia, p on ib:
 *   d   = ((pos_ia - pos_ib) * unit_per_grid + site_offset[orb_site[o]]) - site_offset[orb_site[p]],
 *         then per axis d -= L * rint(d / L), L = box_q * unit_per_grid;   r2 = (dx^2 + dy^2) + dz^2
 *   S   = s_ampl * exp(-0.5 * r2),   H = h_ampl * exp(-sqrt(r2) / h_len)
 *   ia == ib: o == p -> S = 1, H = orb_energy[o];  o != p on the same site -> S = H = 0.
 * eval_fp32 = 0: everything above is evaluated in FP64 with separately rounded operations in exactly that
 * order and the result rounded once to FP32 (so it can differ from a host evaluation only through exp()'s
 * last bit).  eval_fp32 = 1: the paper's choice ("computed in FP32 to make efficient use of
 * the special function units"): FP32 arithmetic from the integer minimum image of the centre difference,
 * __expf; elements then agree with the FP64 evaluation to about 1e-6 absolute.
 * Pairs that are not stored give 0, padding is the identity, as in nolsm_build_submatrices. */
typedef struct {
  const int32_t *pos_q;      /* device [n_mol*3], grid units in [0, box_q) */
  int32_t n_mol;
  int32_t box_q[3];          /* each even */
  int32_t rc_q;
  double unit_per_grid;      /* length of one grid step */
  double site_offset[3][3];  /* [site][axis] */
  int32_t orb_site[6];       /* each in 0..2 */
  double orb_energy[6];
  double s_ampl, h_ampl, h_len;
  int32_t eval_fp32;         /* 0: FP64 evaluation (bit-comparable), 1: FP32 + SFU */
} nolsm_model;

/* Attach (model != NULL; the struct is copied, pos_q stays caller-owned and must outlive its use) or
 * detach (NULL) a model.  While one is attached, every submatrix build of this context --
 * nolsm_build_submatrices and the builds inside nolsm_solve_mu / nolsm_evaluate -- evaluates the model
 * instead of reading H->val and S->val (the pattern arrays are still read; the traces of a6/a7 still
 * read the block stores).  NOLSM_EINVAL for a null pos_q, odd or non-positive box, orb_site out of
 * range, or n_mol different from the matrices' at build time. */
NOLSM_API nolsm_status nolsm_set_model(nolsm_ctx *ctx, const nolsm_model *model /*host*/);

/* How many molecules starting at mol_begin fit in one batch given the workspace bound (host logic;
 * needs row_ptr on the device, synchronises).  Returns the count (>= 0) or -status. */
NOLSM_API int32_t nolsm_batch_capacity(nolsm_ctx *ctx, const nolsm_bsr *H, int32_t mol_begin, int32_t n_slots,
                             void *stream);
NOLSM_API void nolsm_release_batch(nolsm_ctx *ctx, nolsm_batch *batch);

/* a2-a4 (Eq. 15-17, Eq. 12, Eq. 9-10): for every submatrix of the batch, on the first call after the
 * gather: S_j^-1 and B_j = S_j^-1 H_j; on every call: X0 = (B_j - mu I)/s_j with 1.5 s_j >= rho(B_j - mu I)
 * and the sign iteration.  precision/tol/max_iter/fixed_iter < 0 or <= 0 take the context's values.
 * `stats` (host, may be NULL) makes the call synchronise at its end. */
NOLSM_API nolsm_status nolsm_sign_batched(nolsm_ctx *ctx, nolsm_batch *batch, double mu, int32_t precision,
                                float tol, int32_t max_iter, int32_t fixed_iter,
                                nolsm_sign_stats *stats /*host*/, void *stream);

/* a5-a7: D(:, own_j) = 1/2 (I - X_j) S_j^-1(:, own_j) written into rows [mol_begin, ...) of the
 * column-owned store D (same pattern as S), and 2*sum_blocks <D(i,j), S(i,j)>_F of those rows ADDED to
 * *ne_partial (device double; FP32 products, FP64 accumulation).  q_mol (device double [n_mol], may be
 * NULL) receives each molecule's own population; ne_diag (device double, may be NULL) gets
 * sum_j sum_{c in own_j} (1 - X_cc) added.  Asynchronous. */
NOLSM_API nolsm_status nolsm_scatter_density(nolsm_ctx *ctx, const nolsm_batch *batch, const nolsm_bsr *S,
                                   nolsm_bsr *D, double *ne_partial, double *q_mol, double *ne_diag,
                                   void *stream);

/* Whole path (a1-a7) with batching and the bisection of PAPER.md:227: mu = (mu_lo+mu_hi)/2; stop when
 * |N(mu) - n_electrons| <= tol_ne_per_mol * n_mol or after max_steps evaluations (tol_ne_per_mol < 0:
 * always run exactly max_steps evaluations, the timing workload of BASELINE configs[1]);
 * N(mu) > N_e -> mu_hi = mu else mu_lo = mu.  D holds the density of the last evaluated mu.
 * mu_out, ne_out: host doubles.  q_mol: device double [n_mol] or NULL.  Synchronises once per step.
 * The sign iteration stops as nolsm_sign_batched does, but its finishing update X_{k+1} = X_k + 1/2 X_k E_k
 * is applied to the own columns of S_j^-1 only (X_{k+1} V = X_k (V + 1/2 E_k V)) instead of being formed;
 * the iteration counts in the statistics include it (reading 9).
 * The prepare stage (a2, a3) of this call refines what it uses instead of all of S^-1 (reading 11): Eq. 15-17
 * runs on FP16 operands up to its a-priori stop, then B_j and the six own columns of S_j^-1 are refined against S_j
 * once (FP16 mode) or twice (FP32 mode) with the residuals at FP32 quality; the full S_j^-1 does not exist on this
 * path.  The forms nolsm_sign_batched uses are selected by nolsm_config.inv_refine other than 1 (FP16 mode: the
 * refinements then apply to S^-1) and, in FP32 mode, by an explicit inv_refine or inv_tol or by NOLSM_FLAG_NO_PREDICT
 * (Eq. 15-17 itself on split operands to inv_tol). */
NOLSM_API nolsm_status nolsm_solve_mu(nolsm_ctx *ctx, const nolsm_bsr *H, const nolsm_bsr *S, double n_electrons,
                            double mu_lo, double mu_hi, double tol_ne_per_mol, int32_t max_steps,
                            int32_t precision, nolsm_bsr *D, double *mu_out /*host*/,
                            double *ne_out /*host*/, double *q_mol, nolsm_solve_stats *stats /*host*/,
                            void *stream);

/* Energy and energy-weighted density (Eq. 7, 8, 11, 13) of a batch whose sign
 * iterate is current (after nolsm_sign_batched) and whose D columns have been written (nolsm_scatter_density):
 *   W != NULL:        W(:, own_j) = [T_j(D) T_j(H0) T_j(D)](:, own_j) into rows [mol_begin, ...) of the column-owned
 *                     store W (pattern of H; four n x n x 6 products per submatrix, FP32);
 *   e_partial != NULL: sum_j sum_{i in N_j} sum_{o,p} D(i,j)[o,p] H0(j,i)[p,o] ADDED to *e_partial (device double;
 *                     D = the density store; FP32 products, FP64 accumulation).  Asynchronous. */
NOLSM_API nolsm_status nolsm_scatter_energy(nolsm_ctx *ctx, nolsm_batch *batch, const nolsm_bsr *H, const nolsm_bsr *D,
                                  nolsm_bsr *W, double *e_partial, void *stream);

/* One evaluation of the whole path (a1-a7) at a GIVEN mu, plus E_elec = Tr(D H0) (Eq. 7, 11) and, if W != NULL,
 * the energy-weighted density (Eq. 8, 13).  ne_out, e_out: host doubles (N(mu) = 2 tr(DS); E counts every
 * occupied orbital once, as Eq. 7 does).  q_mol: device double [n_mol] or NULL.  Synchronises. */
NOLSM_API nolsm_status nolsm_evaluate(nolsm_ctx *ctx, const nolsm_bsr *H, const nolsm_bsr *S, double mu, int32_t precision,
                            nolsm_bsr *D, nolsm_bsr *W, double *ne_out /*host*/, double *e_out /*host*/,
                            double *q_mol, nolsm_solve_stats *stats /*host*/, void *stream);

/* The same whole path with HOST buffers (the end-to-end call: Fig. 2 d-h of the paper include the
 * transfers).  row_ptr [n_mol+1], col_idx [nnzb], h_val, s_val, d_val [nnzb*36]
 * are HOST pointers (pinned memory makes the copies asynchronous; pageable works).  The context
 * owns device copies of the pattern and of H, S, D (grown on demand, reused across calls); every
 * call copies pattern + H + S host->device, runs nolsm_solve_mu, and copies D device->host.
 * *h2d_bytes / *d2h_bytes (host, may be NULL) receive the bytes moved.  Synchronises. */
NOLSM_API nolsm_status nolsm_solve_mu_host(nolsm_ctx *ctx, int32_t n_mol, const int32_t *row_ptr /*host*/,
                                 const int32_t *col_idx /*host*/, const float *h_val /*host*/,
                                 const float *s_val /*host*/, double n_electrons, double mu_lo,
                                 double mu_hi, double tol_ne_per_mol, int32_t max_steps,
                                 int32_t precision, float *d_val /*host*/, double *mu_out /*host*/,
                                 double *ne_out /*host*/, nolsm_solve_stats *stats /*host*/,
                                 int64_t *h2d_bytes /*host*/, int64_t *d2h_bytes /*host*/, void *stream);

/* Dense microbench entry (BASELINE configs[4]; analogue of the paper's Fig. 6):
 * sign(A_b) for `batch` dense n x n FP32 matrices stored one after another (row-major, leading
 * dimension n).  X0 = A_b / scale[b] (scale: device float [batch], e.g. ||A_b||_2; NULL: the
 * sqrt(||A||_1 ||A||_inf) bound is computed).  x_out: device float [batch*n*n], row-major sign(A_b). */
NOLSM_API nolsm_status nolsm_sign_dense_batched(nolsm_ctx *ctx, const float *a, const float *scale, int32_t n,
                                      int32_t batch, int32_t precision, float tol, int32_t max_iter,
                                      int32_t fixed_iter, float *x_out, nolsm_sign_stats *stats /*host*/,
                                      void *stream);

/* --- the merged pattern of H0 and S ("row i is kept if H_ij != 0 or S_ij != 0") ---
 * The iteration entry points take H and S on ONE pattern.  When the two stores come with different patterns:
 * nolsm_union_pattern (HOST integer work, ascending CSR rows in and out; two passes; NOLSM_ENOMEM with *nnzb_out =
 * needed size when cap is too small) builds the merged pattern, and nolsm_expand_store (device, asynchronous) lays a
 * store out on it: block k of row i = the source's block (i, col_idx_dst[k]) if stored, else zero.  The source
 * pattern must be a subset of the destination's rows-wise (blocks of the source outside it are dropped). */
NOLSM_API nolsm_status nolsm_union_pattern(int32_t n_mol, const int32_t *row_ptr_a /*host*/, const int32_t *col_idx_a /*host*/,
                                           const int32_t *row_ptr_b /*host*/, const int32_t *col_idx_b /*host*/,
                                           int32_t *row_ptr_u /*host [n_mol+1]*/, int32_t *col_idx_u /*host*/, int64_t cap,
                                           int64_t *nnzb_out /*host*/);
NOLSM_API nolsm_status nolsm_expand_store(nolsm_ctx *ctx, const nolsm_bsr *src, const int32_t *row_ptr_dst,
                                          const int32_t *col_idx_dst, float *val_dst, void *stream);

/* --- submatrix combination heuristic (section III-B3, Eq. 14) ---
 * nolsm_combine_submatrices: HOST integer work (the paper runs it on CPU cores, off the clock).
 * Input: the neighbour lists (host CSR, ascending, self included) = the row sets of the one-per-molecule submatrices.
 * Clusters are merged while (n_i + n_j - n_common)^3 < n_i^3 + n_j^3 (Eq. 14); candidates j are the clusters that own
 * a row entry of T_i; they are taken in sweeps over n_{j\i} = |R_j \ R_i| = 0, 1, 2, ...; clusters and candidates in
 * ascending order, T_i updated at once; the sweeps restart until a whole round merges nothing (reading 22).
 * Output (host, caller-allocated): *n_groups_out groups ordered by their smallest owner; own_ptr[n_groups+1] /
 * own_idx[n_mol] = the owners of every group, ascending; list_ptr[n_groups+1] / list_idx = the merged row sets,
 * ascending.  own_ptr and list_ptr need room for n_mol + 1 entries.  If the row sets need more than list_cap
 * entries nothing is written to list_idx and NOLSM_ENOMEM is returned with *list_len_out set to the needed size
 * (it never exceeds the input's nnz).  NOLSM_EINVAL: lists not ascending / out of range, n_mol >= 2^20. */
NOLSM_API nolsm_status nolsm_combine_submatrices(int32_t n_mol, const int32_t *row_ptr /*host*/,
                                                 const int32_t *col_idx /*host*/, int32_t *n_groups_out /*host*/,
                                                 int32_t *own_ptr /*host*/, int32_t *own_idx /*host*/,
                                                 int32_t *list_ptr /*host*/, int32_t *list_idx /*host*/,
                                                 int64_t list_cap, int64_t *list_len_out /*host*/);

typedef struct {            /* the groups on the DEVICE (caller-owned, must outlive the batches built from them) */
  int32_t n_groups;
  const int32_t *own_ptr;   /* [n_groups+1] */
  const int32_t *own_idx;   /* owners (molecules) of every group, ascending */
  const int32_t *list_ptr;  /* [n_groups+1] */
  const int32_t *list_idx;  /* merged row set (molecules) of every group, ascending; contains N_j of every owner j */
} nolsm_groups;

/* Like nolsm_build_submatrices for groups [grp_begin, grp_begin + grp_count): submatrix m of the batch is
 * T(H), T(S) over the merged row set of group grp_begin + m ("common submatrices for multiple similar
 * columns").  nolsm_sign_batched works on it unchanged; nolsm_scatter_density then writes, for every owner j of
 * every group, the blocks D(i, j), i in N_j, from the columns of j inside the combined submatrix (rows of the merged
 * set outside N_j are not stored: the result keeps the pattern of the input) and adds 2 tr(DS) of
 * those owners to *ne_partial.  Gathers from the block stores only (NOLSM_EINVAL while a model is attached). */
NOLSM_API nolsm_status nolsm_build_submatrices_grouped(nolsm_ctx *ctx, const nolsm_bsr *H, const nolsm_bsr *S,
                                                       const nolsm_groups *groups /*host struct*/, int32_t grp_begin,
                                                       int32_t grp_count, int32_t slot, nolsm_batch **out,
                                                       void *stream);

/* Inspection of a batch (tests, parity of the intermediate steps).  which: see NOLSM_MAT_*.
 * Copies submatrix `local` (0-based inside the batch) as a row-major n_j x n_j FP32 matrix into dst
 * (device, capacity dst_elems floats).  *n_out (host) = n_j.  Synchronises. */
#define NOLSM_MAT_S 0     /* T_j(S) as gathered */
#define NOLSM_MAT_H 1     /* T_j(H) as gathered */
#define NOLSM_MAT_SINV 2  /* S_j^-1 (after nolsm_sign_batched) */
#define NOLSM_MAT_B 3     /* B_j = S_j^-1 H_j */
#define NOLSM_MAT_X 4     /* last sign iterate X_j */
NOLSM_API nolsm_status nolsm_batch_read(nolsm_ctx *ctx, const nolsm_batch *batch, int32_t local, int32_t which,
                              float *dst, int64_t dst_elems, int32_t *n_out /*host*/, void *stream);
NOLSM_API int32_t nolsm_batch_size(const nolsm_batch *batch);      /* submatrices in the batch */
NOLSM_API int32_t nolsm_batch_ld(const nolsm_batch *batch);        /* padded leading dimension */

/* One batched product with the engine's own kernels (unit tests of the GEMM building block):
 * C_b = beta*Cin_b + alpha*A_b*B_b (ident = 0)  or  C_b = I - A_b*B_b (ident = 1), b < batch, all
 * n x n row-major FP32 on the device (n arbitrary).  kind: 0 = FP32 SIMT, 1 = tcgen05 FP16 operands,
 * 2 = tcgen05 split-FP16 (FP32-quality), 3 = tcgen05 half-split (A split, B taken as its FP16 rounding: FP32-quality
 * when B is exact in FP16; the add-in travels as a split FP16 pair, 22 bits).  resid2 (device float[batch], may be NULL) receives
 * ||C_b||_F^2 when ident = 1. */
NOLSM_API nolsm_status nolsm_gemm_batched(nolsm_ctx *ctx, int32_t kind, int32_t ident, float alpha, float beta,
                                const float *a, const float *b, const float *cin, float *c,
                                float *resid2, int32_t n, int32_t batch, void *stream);

/* Kernel launches issued by this context so far (bench.py's gpu_launches). */
NOLSM_API int64_t nolsm_launch_count(const nolsm_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* NOLSM_H */
