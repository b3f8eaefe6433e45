// C ABI of libnolsm (include/nolsm.h): context, batching, iteration drivers, mu bisection.
// Host logic only; every arithmetic step of the path runs in the kernels of the other files.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include "common.cuh"

static std::string g_create_err;

#define LAUNCH(ctx, call)                                                                   \
  do {                                                                                      \
    cudaError_t e__ = (call);                                                               \
    (ctx)->launches++;                                                                      \
    if (e__ != cudaSuccess) {                                                               \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);                     \
      return NOLSM_ECUDA;                                                                   \
    }                                                                                       \
  } while (0)

#define CHECK(st)                                  \
  do {                                             \
    nolsm_status s__ = (st);                       \
    if (s__ != NOLSM_OK) return s__;               \
  } while (0)

static int effective_precision(const nolsm_ctx *ctx, int precision) {
  int p = precision < 0 ? ctx->cfg.precision : precision;
  if (ctx->cfg.flags & NOLSM_FLAG_SIMT_ONLY) p = NOLSM_FP32;
  return p;
}

// ------------------------------------------------------------------------------------------------
extern "C" int32_t nolsm_version(void) { return 1; }

extern "C" const char *nolsm_last_error(const nolsm_ctx *ctx) {
  return ctx ? ctx->err.c_str() : g_create_err.c_str();
}

extern "C" int64_t nolsm_launch_count(const nolsm_ctx *ctx) { return ctx ? ctx->launches : 0; }

extern "C" nolsm_status nolsm_create(nolsm_ctx **out, const nolsm_config *cfg) {
  if (!out) return NOLSM_EINVAL;
  *out = nullptr;
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    g_create_err = std::string("no CUDA device: ") + cudaGetErrorString(e);
    cudaGetLastError();
    return NOLSM_ECUDA;
  }
  nolsm_ctx *ctx = new nolsm_ctx();
  nolsm_config c;
  memset(&c, 0, sizeof(c));
  if (cfg) c = *cfg;
  else { c.inv_refine = -1; }
  if (c.precision != NOLSM_FP16_FP32 && c.precision != NOLSM_FP32) { delete ctx; return NOLSM_EINVAL; }
  if (c.max_iter <= 0) c.max_iter = 30;
  if (c.max_iter > NOLSM_MAX_RESID_SLOTS) c.max_iter = NOLSM_MAX_RESID_SLOTS;
  if (c.inv_max_iter <= 0) c.inv_max_iter = 20;
  if (c.inv_max_iter > NOLSM_MAX_RESID_SLOTS) c.inv_max_iter = NOLSM_MAX_RESID_SLOTS;
  ctx->inv_refine_default = c.inv_refine < 0;
  if (c.inv_refine < 0) c.inv_refine = 1;
  if (c.workspace_bytes <= 0) c.workspace_bytes = (int64_t)24 << 30;
  ctx->cfg = c;
  cudaGetDevice(&ctx->device);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, ctx->device) != cudaSuccess) {
    g_create_err = "cudaGetDeviceProperties failed";
    delete ctx;
    return NOLSM_ECUDA;
  }
  ctx->sm_count = prop.multiProcessorCount;
  ctx->l2_bytes = (size_t)prop.l2CacheSize;
  if (cudaMalloc(&ctx->d_scalars, 4 * sizeof(double)) != cudaSuccess ||
      cudaMallocHost(&ctx->h_scalars, 4 * sizeof(double)) != cudaSuccess ||
      cudaMallocHost(&ctx->h_active, NOLSM_MAX_RESID_SLOTS * sizeof(int32_t)) != cudaSuccess) {
    g_create_err = "allocation of context scalars failed";
    delete ctx;
    return NOLSM_ENOMEM;
  }
  for (int i = 0; i < 4; ++i) cudaEventCreateWithFlags(&ctx->ev[i], cudaEventDisableTiming);
  for (int i = 0; i < 2; ++i) cudaEventCreate(&ctx->tev[i]);
  if (prop.major == 10) {
    if (umma_init(ctx) != NOLSM_OK) g_create_err = ctx->err;
  } else {
    ctx->err = "device is not sm_100: tcgen05 path unavailable";
  }
  *out = ctx;
  return NOLSM_OK;
}

static void free_batch(nolsm_batch *b) {
  if (!b) return;
  cudaFree(b->base);
  cudaFree(b->d_dims);
  cudaFree(b->d_state);
  cudaFree(b->d_iters);
  cudaFree(b->d_resid2);
  cudaFree(b->d_lastres);
  cudaFree(b->d_scale);
  cudaFree(b->d_norm);
  cudaFree(b->d_norm_s);
  cudaFree(b->d_scale_s);
  cudaFree(b->d_alpha);
  cudaFree(b->d_colpart);
  cudaFree(b->d_active);
  cudaFree(b->d_tiles_simt);
  cudaFree(b->d_slot_state);
  cudaFree(b->d_slot_done);
  cudaFree(b->d_sched);
  cudaFree(b->d_tile_counter);
  cudaFree(b->d_thin);
  cudaFree(b->d_maps);
  delete b;
}

extern "C" void nolsm_destroy(nolsm_ctx *ctx) {
  if (!ctx) return;
  cudaDeviceSynchronize();
  for (nolsm_batch *b : ctx->slots) free_batch(b);
  cudaFree(ctx->d_scalars);
  cudaFree(ctx->m_row_ptr); cudaFree(ctx->m_col_idx); cudaFree(ctx->m_h); cudaFree(ctx->m_s); cudaFree(ctx->m_d);
  cudaFreeHost(ctx->h_scalars);
  cudaFreeHost(ctx->h_active);
  for (int i = 0; i < 4; ++i)
    if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
  for (int i = 0; i < 2; ++i)
    if (ctx->tev[i]) cudaEventDestroy(ctx->tev[i]);
  delete ctx;
}

extern "C" void nolsm_release_batch(nolsm_ctx *ctx, nolsm_batch *batch) {
  if (!ctx || !batch) return;
  cudaDeviceSynchronize();
  for (size_t i = 0; i < ctx->slots.size(); ++i)
    if (ctx->slots[i] == batch) {
      free_batch(batch);
      ctx->slots[i] = nullptr;
    }
}

extern "C" int32_t nolsm_batch_size(const nolsm_batch *b) { return b ? b->count : 0; }
extern "C" int32_t nolsm_batch_ld(const nolsm_batch *b) { return b ? b->ld : 0; }

// ------------------------------------------------------------------------------------------------
// Batch storage
// ------------------------------------------------------------------------------------------------
// FP32 units per submatrix: S/X, H, Y/S^-1, Z/B and the FP16 operand buffers (two per unit):
// 6 of them in FP16 mode, 10 in FP32 mode (split hi/lo operands); gathered
// batches have four more, the last ones: the split copies of S and H the builder writes.
static int units_dense(int precision) { return precision == NOLSM_FP16_FP32 ? 7 : 9; }
static int units_for(int precision) { return units_dense(precision) + 2; }
static size_t dense_bytes(int count, int ld, int units) {
  return (size_t)units * 4 * (size_t)ld * ld * (size_t)count;
}

// Slots 0..kUserSlots-1 belong to the caller (nolsm_build_submatrices); the whole-path and test entries use
// context-private slots from kOwnSlot on, so that they never invalidate a handle the caller holds.
static const int kUserSlots = 4096;
static const int kOwnSlot = kUserSlots;          // nolsm_solve_mu / nolsm_evaluate / nolsm_solve_mu_host: kOwnSlot + batch
static const int kOwnDense = kUserSlots + 64;    // nolsm_sign_dense_batched, nolsm_gemm_batched

static size_t allocated_bytes(const nolsm_ctx *ctx, int except_slot) {
  size_t t = 0;
  for (size_t i = 0; i < ctx->slots.size(); ++i)
    if (ctx->slots[i] && (int)i != except_slot) t += ctx->slots[i]->base_bytes;
  return t;
}

template <typename T>
static cudaError_t grow(T **ptr, size_t n) {
  cudaFree(*ptr);
  *ptr = nullptr;
  return cudaMalloc(ptr, n * sizeof(T));
}

// Size slot `slot` for `dims` (true dimensions) and upload the metadata.  Host-synchronous uploads
// (small); the dense workspace is grow-only.
static nolsm_status setup_batch(nolsm_ctx *ctx, int slot, const std::vector<int32_t> &dims, int mol_begin,
                                bool sparse, int units, nolsm_batch **out, cudaStream_t st) {
  if (slot < 0 || slot > kOwnDense) { ctx->err = "bad slot"; return NOLSM_EINVAL; }
  if ((int)ctx->slots.size() <= slot) ctx->slots.resize(slot + 1, nullptr);
  if (!ctx->slots[slot]) ctx->slots[slot] = new nolsm_batch();
  nolsm_batch *b = ctx->slots[slot];
  const int count = (int)dims.size();
  int max_n = 0;
  for (int n : dims) max_n = std::max(max_n, n);
  const int ld = std::max(NOLSM_PAD, round_up(max_n, NOLSM_PAD));
  const size_t need = dense_bytes(count, ld, units);
  if (need > b->base_bytes) {
    if ((int64_t)(allocated_bytes(ctx, slot) + need) > ctx->cfg.workspace_bytes) {
      ctx->err = "workspace_bytes too small for this batch";
      return NOLSM_ENOMEM;
    }
    cudaStreamSynchronize(st);
    cudaFree(b->base);
    b->base = nullptr;
    b->base_bytes = 0;
    if (cudaMalloc(&b->base, need) != cudaSuccess) {
      cudaGetLastError();
      ctx->err = "cudaMalloc of the dense workspace failed";
      return NOLSM_ENOMEM;
    }
    b->base_bytes = need;
  }
  if ((size_t)count > b->meta_cap) {
    cudaStreamSynchronize(st);
    const size_t cap = (size_t)count;
    if (grow(&b->d_dims, cap) || grow(&b->d_state, cap) || grow(&b->d_iters, cap) ||
        grow(&b->d_resid2, cap * NOLSM_MAX_RESID_SLOTS) || grow(&b->d_lastres, cap) ||
        grow(&b->d_scale, cap) || grow(&b->d_norm, cap * 2) || grow(&b->d_norm_s, cap * 2) || grow(&b->d_scale_s, cap) || grow(&b->d_alpha, cap * 8) || grow(&b->d_slot_state, cap) ||
        grow(&b->d_slot_done, cap) || grow(&b->d_sched, (size_t)8) || grow(&b->d_tile_counter, (size_t)1) ||
        (b->d_active == nullptr && grow(&b->d_active, (size_t)NOLSM_MAX_RESID_SLOTS))) {
      cudaGetLastError();
      ctx->err = "cudaMalloc of batch metadata failed";
      return NOLSM_ENOMEM;
    }
    b->meta_cap = cap;
  }
  {
    const size_t need_cp = (size_t)count * colpart_strips(ld) * ld;
    if (need_cp > b->colpart_cap) {
      cudaStreamSynchronize(st);
      if (grow(&b->d_colpart, need_cp)) { cudaGetLastError(); ctx->err = "cudaMalloc of the norm scratch failed"; return NOLSM_ENOMEM; }
      b->colpart_cap = need_cp;
    }
  }
  NOLSM_CUDA(ctx, cudaMemsetAsync(b->d_sched, 0, 8 * sizeof(int32_t), st));
  b->count = count;
  b->s32_built = true;
  b->s_norm_built = false;
  b->sinv_own_only = false;
  b->x0_built = false;
  b->b32_built = true;
  b->lowdin = false;
  b->ld = ld;
  b->max_n = max_n;
  b->mol_begin = mol_begin;
  b->slot = slot;
  b->sparse = sparse;
  b->prepared = false;
  b->prepared_precision = -1;
  const bool unit_scale = (ctx->cfg.flags & NOLSM_FLAG_UNIT_SCALE) != 0;
  b->inv_scale = unit_scale ? 1.f : 0.5f;
  b->sign_scale = unit_scale ? 1.f : 1.f / 1.5f;
  b->n_host = dims;
  b->n_unit = units;
  b->n_half = 2 * (units - 4);
  const size_t slab = (size_t)ld * ld;
  for (int i = 0; i < units; ++i) b->u[i] = reinterpret_cast<float *>(b->base) + (size_t)i * count * slab;
  for (int i = 0; i < b->n_half; ++i) b->h[i] = reinterpret_cast<__half *>(b->u[4]) + (size_t)i * count * slab;
  // tile list of the SIMT kernel (debug path); the tcgen05 engine enumerates its tiles arithmetically
  std::vector<TileDesc> tiles_simt;
  b->sum_n3 = b->sum_n3_padded = 0.0;
  const bool simt = (ctx->cfg.flags & NOLSM_FLAG_SIMT_ONLY) != 0 || !ctx->umma_ok || !sparse;
  for (int m = 0; m < count; ++m) {
    const int n = dims[m];
    const int P = round_up(n, NOLSM_TILE_M), Pn = round_up(n, 16);
    if (simt)
      for (int n0 = 0; n0 < P; n0 += 128)
        for (int m0 = 0; m0 < P; m0 += 128) tiles_simt.push_back(TileDesc{m, m0, n0, 128});
    b->sum_n3 += (double)n * n * n;
    b->sum_n3_padded += (double)P * Pn * Pn;
  }
  if (tiles_simt.size() > b->tiles_simt_cap) {
    cudaStreamSynchronize(st);
    if (grow(&b->d_tiles_simt, tiles_simt.size())) { cudaGetLastError(); ctx->err = "cudaMalloc tiles"; return NOLSM_ENOMEM; }
    b->tiles_simt_cap = tiles_simt.size();
  }
  b->n_tiles_simt = (int)tiles_simt.size();
  {
    double p128 = 0.0, p256 = 0.0, sum_n = 0.0;
    for (int n : dims) { p128 += round_up(n, 128); p256 += round_up(n, 256); sum_n += n; }
    b->prefer_pair = count > 0 && sum_n >= 1100.0 * count && p256 <= 1.04 * p128;
  }
  // pageable host buffers: cudaMemcpyAsync stages them before returning, so the vectors may die
  NOLSM_CUDA(ctx, cudaMemcpyAsync(b->d_dims, dims.data(), sizeof(int32_t) * count, cudaMemcpyHostToDevice, st));
  if (!tiles_simt.empty())
    NOLSM_CUDA(ctx, cudaMemcpyAsync(b->d_tiles_simt, tiles_simt.data(), sizeof(TileDesc) * tiles_simt.size(),
                                    cudaMemcpyHostToDevice, st));
  NOLSM_CUDA(ctx, cudaStreamSynchronize(st));
  CHECK(umma_make_maps(ctx, b));
  *out = b;
  return NOLSM_OK;
}

// ------------------------------------------------------------------------------------------------
// a0
// ------------------------------------------------------------------------------------------------
extern "C" nolsm_status nolsm_build_neighbours(nolsm_ctx *ctx, int32_t n_mol, const int32_t *pos_q,
                                               const int32_t *box_q, int32_t rc_q, int32_t *row_ptr,
                                               int32_t *col_idx, int64_t cap, int64_t *nnzb_out, void *stream) {
  if (!ctx) return NOLSM_EINVAL;
  if (n_mol < 0 || !row_ptr || !box_q || (n_mol > 0 && !pos_q) || rc_q < 0 || cap < 0) {
    ctx->err = "nolsm_build_neighbours: bad argument";
    return NOLSM_EINVAL;
  }
  for (int a = 0; a < 3; ++a)
    if (box_q[a] <= 0 || (box_q[a] & 1)) { ctx->err = "box lengths must be positive and even"; return NOLSM_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  int32_t *counts = nullptr;
  NOLSM_CUDA(ctx, cudaMalloc(&counts, sizeof(int32_t) * std::max(n_mol, 1)));
  cudaError_t e = launch_neighbour_count(n_mol, pos_q, box_q, rc_q, counts, st);
  ctx->launches++;
  if (e == cudaSuccess) { e = launch_exclusive_scan(counts, row_ptr, n_mol, st); ctx->launches++; }
  int32_t total = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&total, row_ptr + n_mol, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(counts);
  if (e != cudaSuccess) { ctx->err = std::string("neighbour count: ") + cudaGetErrorString(e); return NOLSM_ECUDA; }
  if (nnzb_out) *nnzb_out = total;
  if ((int64_t)total > cap || (total > 0 && !col_idx)) {
    ctx->err = "col_idx capacity too small";
    return NOLSM_ENOMEM;
  }
  LAUNCH(ctx, launch_neighbour_fill(n_mol, pos_q, box_q, rc_q, row_ptr, col_idx, st));
  return NOLSM_OK;
}

// ------------------------------------------------------------------------------------------------
// a1
// ------------------------------------------------------------------------------------------------
static nolsm_status check_bsr(nolsm_ctx *ctx, const nolsm_bsr *m, const char *name) {
  if (!m || m->bs != NOLSM_BS || m->n_mol < 0 || !m->row_ptr || (m->n_mol > 0 && (!m->col_idx || !m->val))) {
    ctx->err = std::string("bad block-sparse matrix ") + name + " (bs must be 6, pointers non-null)";
    return NOLSM_EINVAL;
  }
  if (reinterpret_cast<uintptr_t>(m->val) & 15) {   // the gather reads pairs of block rows with 16-byte loads
    ctx->err = std::string("block-sparse matrix ") + name + ": val must be 16-byte aligned";
    return NOLSM_EINVAL;
  }
  return NOLSM_OK;
}

static nolsm_status read_dims(nolsm_ctx *ctx, const int32_t *row_ptr, int mol_begin, int mol_count,
                              std::vector<int32_t> &dims, cudaStream_t st) {
  std::vector<int32_t> rp(mol_count + 1);
  NOLSM_CUDA(ctx, cudaMemcpyAsync(rp.data(), row_ptr + mol_begin, sizeof(int32_t) * (mol_count + 1),
                                  cudaMemcpyDeviceToHost, st));
  NOLSM_CUDA(ctx, cudaStreamSynchronize(st));
  dims.resize(mol_count);
  for (int i = 0; i < mol_count; ++i) {
    dims[i] = (rp[i + 1] - rp[i]) * NOLSM_BS;
    if (dims[i] <= 0) { ctx->err = "molecule with an empty neighbour list (self must be included)"; return NOLSM_EINVAL; }
  }
  return NOLSM_OK;
}

extern "C" int32_t nolsm_batch_capacity(nolsm_ctx *ctx, const nolsm_bsr *H, int32_t mol_begin, int32_t n_slots,
                                        void *stream) {
  if (!ctx || check_bsr(ctx, H, "H") != NOLSM_OK || mol_begin < 0 || mol_begin > H->n_mol || n_slots <= 0)
    return -(int32_t)NOLSM_EINVAL;
  const int avail = H->n_mol - mol_begin;
  if (avail == 0) return 0;
  std::vector<int32_t> dims;
  nolsm_status s = read_dims(ctx, H->row_ptr, mol_begin, avail, dims, (cudaStream_t)stream);
  if (s != NOLSM_OK) return -(int32_t)s;
  const size_t budget = (size_t)ctx->cfg.workspace_bytes / (size_t)n_slots;
  const int units = units_for(effective_precision(ctx, -1));
  int max_n = 0, count = 0;
  for (int i = 0; i < avail; ++i) {
    const int mn = std::max(max_n, dims[i]);
    if (dense_bytes(i + 1, round_up(mn, NOLSM_PAD), units) > budget) break;
    max_n = mn;
    count = i + 1;
  }
  return count;
}

extern "C" nolsm_status nolsm_set_model(nolsm_ctx *ctx, const nolsm_model *model) {
  if (!ctx) return NOLSM_EINVAL;
  if (!model) { ctx->has_model = false; return NOLSM_OK; }
  if (!model->pos_q || model->n_mol <= 0 || model->rc_q < 0 || !(model->unit_per_grid > 0.0) ||
      !(model->h_len > 0.0)) {
    ctx->err = "model: null positions, empty system, negative cutoff or non-positive length scale";
    return NOLSM_EINVAL;
  }
  for (int i = 0; i < 3; ++i)
    if (model->box_q[i] <= 0 || (model->box_q[i] & 1)) { ctx->err = "model: box_q must be positive and even"; return NOLSM_EINVAL; }
  for (int o = 0; o < NOLSM_BS; ++o)
    if (model->orb_site[o] < 0 || model->orb_site[o] > 2) { ctx->err = "model: orb_site must be 0, 1 or 2"; return NOLSM_EINVAL; }
  ctx->model = *model;
  ctx->has_model = true;
  return NOLSM_OK;
}

static nolsm_status build_submatrices_impl(nolsm_ctx *ctx, const nolsm_bsr *H, const nolsm_bsr *S,
                                           int32_t mol_begin, int32_t mol_count, int32_t slot, int units,
                                           nolsm_batch **out, void *stream, bool need_h32 = true,
                                           bool need_s32 = true, bool fast32 = false) {
  if (!ctx || !out) return NOLSM_EINVAL;
  CHECK(check_bsr(ctx, H, "H"));
  CHECK(check_bsr(ctx, S, "S"));
  if (H->n_mol != S->n_mol || H->row_ptr != S->row_ptr || H->col_idx != S->col_idx) {
    ctx->err = "H and S must share one pattern (row_ptr, col_idx)";
    return NOLSM_EINVAL;
  }
  if (mol_begin < 0 || mol_count < 0 || mol_begin + mol_count > H->n_mol) {
    ctx->err = "molecule range outside the matrix";
    return NOLSM_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)stream;
  std::vector<int32_t> dims;
  if (mol_count > 0) CHECK(read_dims(ctx, H->row_ptr, mol_begin, mol_count, dims, st));
  nolsm_batch *b = nullptr;
  CHECK(setup_batch(ctx, slot, dims, mol_begin, true, units, &b, st));
  // the split copy of S is only read by the Newton refinements of S^-1 (reading 11)
  const int prec = effective_precision(ctx, -1);
  // (fast32: the whole path's FP32 mode runs the FP16 chain and refines twice, prepare_batch_chain)
  const bool split_s = fast32 || (ctx->cfg.inv_refine >= 0 ? ctx->cfg.inv_refine : (prec == NOLSM_FP16_FP32 ? 1 : 0)) > 0;
  // the FP32 copy of T_j(S) can only be left out where the lean FP16 start of Eq. 15-17 reads the split copy
  if (!(split_s && (prec == NOLSM_FP16_FP32 || fast32)) || ctx->has_model) need_s32 = true;
  b->s_norm_built = false;
  if (ctx->has_model) {
    if (ctx->model.n_mol != H->n_mol) {
      ctx->err = "the attached model has a different number of molecules than the matrices";
      return NOLSM_EINVAL;
    }
    LAUNCH(ctx, launch_generate(b, H->row_ptr, H->col_idx, &ctx->model, need_h32 ? b->u[1] : nullptr, b->u[0],
                                split_s, st));
  } else {
    // the builder sees every column of T_j(S) whole: its norm bound comes out of the same pass
    NOLSM_CUDA(ctx, cudaMemsetAsync(b->d_norm_s, 0, sizeof(float) * 2 * b->count, st));
    LAUNCH(ctx, launch_gather(b, H->row_ptr, H->col_idx, nullptr, nullptr, H->val, S->val,
                              need_h32 ? b->u[1] : nullptr, need_s32 ? b->u[0] : nullptr, split_s, b->d_norm_s, st));
    b->s_norm_built = true;
  }
  b->s_split_built = split_s;
  b->s32_built = need_s32;
  b->row_ptr = H->row_ptr;
  b->col_idx = H->col_idx;
  b->grouped = false;
  *out = b;
  return NOLSM_OK;
}

// The merged H0 u S pattern: a store re-laid on the union pattern of nolsm_union_pattern.
extern "C" nolsm_status nolsm_expand_store(nolsm_ctx *ctx, const nolsm_bsr *src, const int32_t *row_ptr_dst,
                                           const int32_t *col_idx_dst, float *val_dst, void *stream) {
  if (!ctx) return NOLSM_EINVAL;
  CHECK(check_bsr(ctx, src, "src"));
  if (!row_ptr_dst || (src->n_mol > 0 && (!col_idx_dst || !val_dst))) { ctx->err = "nolsm_expand_store: null destination"; return NOLSM_EINVAL; }
  LAUNCH(ctx, launch_expand_store(src->n_mol, src->row_ptr, src->col_idx, src->val, row_ptr_dst, col_idx_dst, val_dst,
                                  (cudaStream_t)stream));
  return NOLSM_OK;
}

// a batch of COMBINED submatrices.  Group g's dense pair is T(H), T(S) over its
// merged row set; everything downstream of the gather (Eq. 15-17, sign iteration) is the same batch machinery.
extern "C" nolsm_status nolsm_build_submatrices_grouped(nolsm_ctx *ctx, const nolsm_bsr *H, const nolsm_bsr *S,
                                                        const nolsm_groups *groups, int32_t grp_begin,
                                                        int32_t grp_count, int32_t slot, nolsm_batch **out,
                                                        void *stream) {
  if (!ctx || !out || !groups) return NOLSM_EINVAL;
  CHECK(check_bsr(ctx, H, "H"));
  CHECK(check_bsr(ctx, S, "S"));
  if (slot < 0 || slot >= kUserSlots) { ctx->err = "slot must be in [0, 4096)"; return NOLSM_EINVAL; }
  if (H->n_mol != S->n_mol || H->row_ptr != S->row_ptr || H->col_idx != S->col_idx) {
    ctx->err = "H and S must share one pattern (row_ptr, col_idx)";
    return NOLSM_EINVAL;
  }
  if (!groups->own_ptr || !groups->own_idx || !groups->list_ptr || !groups->list_idx || grp_begin < 0 ||
      grp_count < 0 || grp_begin + grp_count > groups->n_groups) {
    ctx->err = "bad group arrays or group range";
    return NOLSM_EINVAL;
  }
  if (ctx->has_model) { ctx->err = "combined submatrices are gathered from the block stores (detach the model)"; return NOLSM_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  std::vector<int32_t> lp(grp_count + 1), op(grp_count + 1), dims(grp_count);
  if (grp_count > 0) {
    NOLSM_CUDA(ctx, cudaMemcpyAsync(lp.data(), groups->list_ptr + grp_begin, sizeof(int32_t) * (grp_count + 1),
                                    cudaMemcpyDeviceToHost, st));
    NOLSM_CUDA(ctx, cudaMemcpyAsync(op.data(), groups->own_ptr + grp_begin, sizeof(int32_t) * (grp_count + 1),
                                    cudaMemcpyDeviceToHost, st));
    NOLSM_CUDA(ctx, cudaStreamSynchronize(st));
  }
  for (int i = 0; i < grp_count; ++i) {
    dims[i] = (lp[i + 1] - lp[i]) * NOLSM_BS;
    if (dims[i] <= 0 || op[i + 1] <= op[i]) { ctx->err = "group with an empty row set or without an owner"; return NOLSM_EINVAL; }
  }
  nolsm_batch *b = nullptr;
  const int prec = effective_precision(ctx, -1);
  CHECK(setup_batch(ctx, slot, dims, grp_begin, true, units_for(prec), &b, st));
  const bool split_s = (ctx->cfg.inv_refine >= 0 ? ctx->cfg.inv_refine : (prec == NOLSM_FP16_FP32 ? 1 : 0)) > 0;
  LAUNCH(ctx, launch_gather(b, H->row_ptr, H->col_idx, groups->list_ptr, groups->list_idx, H->val, S->val, b->u[1],
                            b->u[0], split_s, nullptr, st));
  b->s_split_built = split_s;
  b->row_ptr = H->row_ptr;
  b->col_idx = H->col_idx;
  b->grouped = true;
  b->g_own_ptr = groups->own_ptr; b->g_own_idx = groups->own_idx;
  b->g_list_ptr = groups->list_ptr; b->g_list_idx = groups->list_idx;
  b->own_first = grp_count > 0 ? op[0] : 0;
  b->own_count = grp_count > 0 ? op[grp_count] - op[0] : 0;
  *out = b;
  return NOLSM_OK;
}

extern "C" nolsm_status nolsm_build_submatrices(nolsm_ctx *ctx, const nolsm_bsr *H, const nolsm_bsr *S,
                                                int32_t mol_begin, int32_t mol_count, int32_t slot,
                                                nolsm_batch **out, void *stream) {
  if (!ctx) return NOLSM_EINVAL;
  if (slot < 0 || slot >= kUserSlots) { ctx->err = "slot must be in [0, 4096)"; return NOLSM_EINVAL; }
  return build_submatrices_impl(ctx, H, S, mol_begin, mol_count, slot, units_for(effective_precision(ctx, -1)), out,
                                stream);
}

// ------------------------------------------------------------------------------------------------
// Iteration drivers
// ------------------------------------------------------------------------------------------------
static bool use_simt(const nolsm_ctx *ctx) { return (ctx->cfg.flags & NOLSM_FLAG_SIMT_ONLY) != 0; }

static int group_size(const nolsm_ctx *ctx, const nolsm_batch *b, int bytes_per_elem) {
  if (ctx->cfg.group > 0) return ctx->cfg.group;
  // Two pulls: the iterates of a group should stay in L2 over an iteration,
  // and dependent products must be far apart in the claim order, or CTAs idle on the dependency flags.
  // Measured on w32768 (bench.py --group): 8 -> 582, 14 -> 652, 24 -> 698, 40 -> 703, 96 -> 697 TFLOP/s:
  // the distance matters more than the residency, so a group holds at least eight waves of tiles.
  const double per = (double)bytes_per_elem * b->ld * b->ld;
  int g = (int)(0.75 * (double)ctx->l2_bytes / per);
  const int tiles = std::max(1, ((b->max_n + 127) / 128) * ((b->max_n + 255) / 256));
  const int g_min = (8 * ctx->sm_count + tiles - 1) / tiles;
  g = std::max(g, g_min);
  return std::max(1, std::min(g, 1024));
}

static ChainOp make_op(int mode, float alpha, float beta) {
  ChainOp o;
  memset(&o, 0, sizeof(o));
  for (int p = 0; p < 2; ++p) o.a[p] = o.b[p] = o.a_lo[p] = o.b_lo[p] = o.out16[p] = o.out16_lo[p] = -1;
  o.cin32 = o.cout32 = -1;
  o.cin16[0] = o.cin16[1] = -1;
  o.cin16_lo[0] = o.cin16_lo[1] = -1;
  o.mode = mode;
  o.alpha = alpha;
  o.beta = beta;
  return o;
}
static void set2(int32_t (&d)[2], int even, int odd) { d[0] = even; d[1] = odd; }

static nolsm_status run_chain(nolsm_ctx *ctx, nolsm_batch *b, const ChainProgram &pg, const float *alpha_div,
                              bool touch_stats, cudaStream_t st) {
  cudaError_t e = launch_chain(ctx, b, pg, alpha_div, touch_stats, st);
  ctx->launches += 2;   // reset kernel + chain kernel
  if (e != cudaSuccess) {
    ctx->err = std::string("tcgen05 chain: ") + cudaGetErrorString(e) +
               (ctx->umma_ok ? "" : " (tcgen05 path not initialised: needs an sm_100 device)");
    cudaGetLastError();
    return NOLSM_ECUDA;
  }
  return NOLSM_OK;
}

static nolsm_status join_sinv(nolsm_ctx *ctx, nolsm_batch *b, cudaStream_t st);

static ChainProgram one_shot(int group) {
  ChainProgram pg;
  memset(&pg, 0, sizeof(pg));
  pg.max_iter = 1;
  pg.fixed_iter = 1;
  pg.group = group;
  return pg;
}

// a2 + a3 (first part) on the tensor cores: S^-1 by Eq. 15-17 in the correction
// form  E = I - Z Y,  Y += 1/2 Y E,  Z += 1/2 E Z  (= Eq. 16 with 3I - V = 2I + E), then
// S^-1 = Z^2 / s_S (Eq. 17), optional Newton refinements (reading 11) and B = S^-1 H
// (Eq. 12).  FP16 mode: the iteration runs on plain FP16 operands, everything after it
// on split (hi + lo) operands; FP32 mode: every product on split operands.
static nolsm_status ensure_thin(nolsm_ctx *ctx, nolsm_batch *b, cudaStream_t st);

// own_only (nolsm_solve_mu without energy products: nothing downstream reads S^-1 outside its six own columns):
// the refinement is applied to B and to those columns instead of to all of S^-1, see below.
// x0_mu (with own_only): the chemical potential of the ONE sign evaluation that will follow -- B is then never
// written; B1's epilogue emits X0 = (B1 - mu I)/s_j as the split pair the sign iteration starts from.
static nolsm_status prepare_batch_chain(nolsm_ctx *ctx, nolsm_batch *b, int precision, cudaStream_t st,
                                        nolsm_sign_stats *stats, int64_t *gemms, bool own_only,
                                        const double *x0_mu) {
  // FP32 mode of the whole path (defaults only): the same FP16 chain and A0, then TWO refinements of B and of the own
  // columns of S^-1 -- with F = I - A0 S the errors are F^3 B and F^3 V, ||F||_2 <= 1e-2 by the a-priori stop, and the
  // residuals are formed on split operands -- instead of running Eq. 15-17 itself on split operands to 1e-5:
  // 14 MMA-equivalents instead of about 30.  Below, `fp16` then selects the FP16 chain and buffer layout.
  // Loewdin form (NOLSM_FLAG_LOWDIN; nolsm_solve_mu checked the precision): Eq. 15-17 on split operands to its end
  const bool lowdin = own_only && (ctx->cfg.flags & NOLSM_FLAG_LOWDIN) != 0 && precision != NOLSM_FP16_FP32 &&
                      b->sparse && b->row_ptr != nullptr && !b->grouped;
  b->lowdin = false;
  const bool fp32_fast = !lowdin && precision != NOLSM_FP16_FP32 && own_only && ctx->inv_refine_default && ctx->cfg.inv_tol <= 0.f &&
                         (ctx->cfg.flags & NOLSM_FLAG_NO_PREDICT) == 0 && b->sparse && b->row_ptr != nullptr &&
                         !b->grouped && b->s_split_built && b->s_norm_built;
  const bool fp16 = precision == NOLSM_FP16_FP32 || fp32_fast;
  const int refine = lowdin ? 0 : (fp32_fast ? 1 : (ctx->cfg.inv_refine >= 0 ? ctx->cfg.inv_refine : (fp16 ? 1 : 0)));
  // one refinement, FP16 mode, one owner per submatrix: B1 = B0 + A0 (H - S B0) with B0 = A0 H and A0 = Z^2/s_S the
  // FP16-quality inverse -- the same second-order error (I - A0 S)^2 S^-1 H as refining S^-1 first, in four MMAs
  // (1 + 2 + 1) instead of seven (3 + 1 for the refinement, 3 for B on split operands); the own columns of S^-1
  // get their refinement as two thin products (launch_own_refine)
  const bool fast_b = own_only && fp16 && refine == 1 && b->sparse && b->row_ptr != nullptr && !b->grouped;
  const bool x0_direct = fast_b && !fp32_fast && x0_mu != nullptr && (ctx->cfg.flags & NOLSM_FLAG_ORDER3) == 0;
  b->x0_built = false;
  b->b32_built = true;
  // 3e-3 with a refinement behind: the iterate is taken with a relative error of about twice its residual,
  // which the refinement squares (< 4e-5)
  const float inv_tol = ctx->cfg.inv_tol > 0.f ? ctx->cfg.inv_tol : (fp16 ? (refine > 0 ? 3e-3f : 1e-2f) : 1e-5f);
  float *S = b->u[0], *H = b->u[1];
  // FP16 mode with a refinement behind the iteration: the iterates live in FP16 only (the add-in of the
  // correction form is the FP16 operand copy itself); their 5e-4 rounding is far inside what the refinement
  // squares away, and no tile reads or writes an FP32 master
  const bool masters = !(fp16 && refine > 0);
  // lean start: the builder left the split copy of S and its norm bound; Y0 is never written (launch_init_z1)
  const bool lean = !masters && b->s_split_built && b->s_norm_built;
  if (!lean && !b->s32_built) { ctx->err = "this batch was built without the FP32 copy of S"; return NOLSM_EINVAL; }
  const float *s_norm = b->s_norm_built ? b->d_norm_s : b->d_norm;
  if (!b->s_norm_built) LAUNCH(ctx, launch_norm_bound(b, S, 0.f, true, b->d_norm, st));
  ChainProgram pg;
  memset(&pg, 0, sizeof(pg));
  pg.n_ops = 3;
  pg.max_iter = ctx->cfg.inv_max_iter;
  pg.fixed_iter = 0;
  pg.tol = inv_tol;
  // Iteration 0 in closed form (Z0 = I): E0 = I - Y0, Z1 = 3/2 I - 1/2 Y0 element-wise, Y1 = Y0 + 1/2 Y0 E0 by
  // one product; the chain then starts at iteration 1, i.e. on the odd-parity buffers.
  pg.max_iter = std::max(1, ctx->cfg.inv_max_iter - 1);
  // With a Newton refinement behind it (which squares the error) the iterate whose residual passes the
  // test is taken as it is: the two products that would finish that iteration are skipped (reading 11).
  pg.stop_early = refine > 0 ? 1 : 0;
  ChainProgram p0 = one_shot(group_size(ctx, b, 16));
  p0.n_ops = 1;
  ChainOp &y1 = p0.ops[0] = make_op(EPI_AXPBY, 0.5f, 1.f);
  y1.cin32 = y1.cout32 = 2;
  if (fp16) {
    // Y16: h0/h1 (ping-pong), Z16: h2/h3, E16: h4; masters (if kept) Y32 = u2, Z32 = u3
    if (lean)
      LAUNCH(ctx, launch_init_z1(b, b->h[b->n_half - 4], b->h[b->n_half - 3], s_norm, b->h[3], b->d_scale, st));
    else
      LAUNCH(ctx, launch_init_inverse_first(b, S, s_norm, masters ? b->u[2] : nullptr, masters ? b->u[3] : nullptr,
                                            b->h[0], nullptr, b->h[3], nullptr, b->h[4], nullptr, b->d_scale, st));
    set2(y1.a, 0, 0); set2(y1.b, 4, 4); set2(y1.out16, 1, 1);
    pg.group = group_size(ctx, b, masters ? 18 : 10);
    ChainOp &e = pg.ops[0] = make_op(EPI_IDENT, 1.f, 0.f);
    set2(e.a, 3, 2); set2(e.b, 1, 0); set2(e.out16, 4, 4); e.resid = 1;
    // Z before Y (they are independent given E): an a-priori stop ends the submatrix after the Z update
    ChainOp &z = pg.ops[1] = make_op(EPI_AXPBY, 0.5f, 1.f);
    set2(z.a, 4, 4); set2(z.b, 3, 2); z.cin32 = z.cout32 = 3; set2(z.out16, 2, 3);
    ChainOp &y = pg.ops[2] = make_op(EPI_AXPBY, 0.5f, 1.f);
    set2(y.a, 1, 0); set2(y.b, 4, 4); y.cin32 = y.cout32 = 2; set2(y.out16, 0, 1);
    pg.skip_tail = 1;   // without stop_early: the iteration that ends the chain does not form Y_{k+1}
    if (pg.stop_early && (ctx->cfg.flags & NOLSM_FLAG_NO_PREDICT) == 0) {
      // a-priori stop (ChainProgram::tol_pred, reading 11): ||E_{k+1}||_2 <= 2e-2 guaranteed from ||E_k||_1,
      // i.e. a relative error of at most 2e-2 in every direction of A0, which the refinement squares
      e.colnorm = 1;
      pg.tol_pred = fp32_fast ? 1e-2f : 2e-2f;
    }
    if (lean) {   // Y1 = Y0 Z1 = (S_hi Z1)/s_S: plain product, scaled in the epilogue
      y1 = make_op(EPI_AXPBY, 1.f, 0.f);
      y1.use_div = 1;
      set2(y1.a, b->n_half - 4, b->n_half - 4); set2(y1.b, 3, 3); set2(y1.out16, 1, 1);
    }
    if (!masters) {
      if (!lean) { y1.cin32 = y1.cout32 = -1; set2(y1.cin16, 0, 0); }
      y.cin32 = y.cout32 = -1; set2(y.cin16, 1, 0);
      z.cin32 = z.cout32 = -1; set2(z.cin16, 3, 2);
    }
  } else {
    // split operands: Y (h0,h1)/(h2,h3), Z (h4,h5)/(h6,h7), E (h8,h9)
    // the iterates live as split pairs only (22 bits): the add-in of the correction form is the operand pair itself
    LAUNCH(ctx, launch_init_inverse_first(b, S, s_norm, nullptr, nullptr, b->h[0], b->h[1], b->h[6], b->h[7],
                                          b->h[8], b->h[9], b->d_scale, st));
    set2(y1.a, 0, 0); set2(y1.a_lo, 1, 1); set2(y1.b, 8, 8); set2(y1.b_lo, 9, 9);
    set2(y1.out16, 2, 2); set2(y1.out16_lo, 3, 3);
    y1.cin32 = y1.cout32 = -1; set2(y1.cin16, 0, 0); set2(y1.cin16_lo, 1, 1);
    pg.group = group_size(ctx, b, 28);
    ChainOp &e = pg.ops[0] = make_op(EPI_IDENT, 1.f, 0.f);
    set2(e.a, 6, 4); set2(e.a_lo, 7, 5); set2(e.b, 2, 0); set2(e.b_lo, 3, 1);
    set2(e.out16, 8, 8); set2(e.out16_lo, 9, 9); e.resid = 1;
    // Z before Y: the iteration that ends the chain does not form Y_{k+1} (nothing reads it)
    ChainOp &z = pg.ops[1] = make_op(EPI_AXPBY, 0.5f, 1.f);
    set2(z.a, 8, 8); set2(z.a_lo, 9, 9); set2(z.b, 6, 4); set2(z.b_lo, 7, 5);
    set2(z.cin16, 6, 4); set2(z.cin16_lo, 7, 5); set2(z.out16, 4, 6); set2(z.out16_lo, 5, 7);
    ChainOp &y = pg.ops[2] = make_op(EPI_AXPBY, 0.5f, 1.f);
    set2(y.a, 2, 0); set2(y.a_lo, 3, 1); set2(y.b, 8, 8); set2(y.b_lo, 9, 9);
    set2(y.cin16, 2, 0); set2(y.cin16_lo, 3, 1); set2(y.out16, 0, 2); set2(y.out16_lo, 1, 3);
    pg.skip_tail = 1;
  }
  CHECK(run_chain(ctx, b, p0, lean ? b->d_scale : nullptr, false, st));
  CHECK(run_chain(ctx, b, pg, nullptr, true, st));
  // submatrices whose Eq. 15-17 iteration ended at the cap or on a NaN (S_j not SPD / badly scaled): kept beside
  // the scheduler words, which the next launch resets
  NOLSM_CUDA(ctx, cudaMemcpyAsync(b->d_sched + 4, b->d_sched + 2, sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
  int64_t inv_gemm_sum = 0;
  if (stats) {   // iterations and residuals of Eq. 15-17, before the sign iteration reuses the arrays
    std::vector<int32_t> it(b->count);
    std::vector<float> res(b->count);
    NOLSM_CUDA(ctx, cudaMemcpyAsync(it.data(), b->d_iters, sizeof(int32_t) * b->count, cudaMemcpyDeviceToHost, st));
    NOLSM_CUDA(ctx, cudaMemcpyAsync(res.data(), b->d_lastres, sizeof(float) * b->count, cudaMemcpyDeviceToHost, st));
    std::vector<int32_t> how(b->count);   // state word of the chain: last op of the stopping iteration << 24
    NOLSM_CUDA(ctx, cudaMemcpyAsync(how.data(), b->d_state, sizeof(int32_t) * b->count, cudaMemcpyDeviceToHost, st));
    NOLSM_CUDA(ctx, cudaStreamSynchronize(st));
    double fl = 0.0;
    for (int m = 0; m < b->count; ++m) {
      // chain iterations carried out in full; a stop_early chain ran one residual product more; one that stopped
      // a priori ran E and Z of its last iteration only
      const bool ahead = ((how[m] >> 24) & 0x7f) == 1 && how[m] != 0x7fffffff;
      const int chain_products = ahead ? 3 * it[m] - 1 : 3 * it[m] + pg.stop_early - (pg.stop_early ? 0 : pg.skip_tail);
      it[m] += 1;   // iteration 0 ran in closed form
      stats->inv_iter_max = std::max(stats->inv_iter_max, it[m]);
      if (!(res[m] <= stats->inv_worst_residual)) stats->inv_worst_residual = res[m];
      const double n = b->n_host[m];
      const int products = 1 + chain_products + 2 + 2 * refine + (fp32_fast ? 2 : 0);   // products, whatever the MMAs per product
      inv_gemm_sum += products;
      fl += 2.0 * n * n * n * products;
    }
    stats->flops_prepare = fl;
  }
  const int g1 = group_size(ctx, b, 16);
  if (lowdin) {
    // Z = (S / s_S)^-1/2 is the chain's last Z iterate, in (h4,h5) or (h6,h7) by parity: make it (h6,h7) for all, which
    // the sign iteration (h0..h5) leaves alone.  T = H Z -> (h8,h9);  A~ = Z T / s_S -> u3 (symmetric);
    // Z[:, own] -> FP32 own columns of u2 (where a5 looks for its thin operand); s_S kept for a5.
    LAUNCH(ctx, launch_canon_pair(b, b->d_iters, b->h[4], b->h[5], b->h[6], b->h[7], st));
    NOLSM_CUDA(ctx, cudaMemcpyAsync(b->d_scale_s, b->d_scale, sizeof(float) * b->count, cudaMemcpyDeviceToDevice, st));
    const int hh = b->n_half - 2, hl = b->n_half - 1;
    ChainProgram pt = one_shot(g1);
    pt.n_ops = 1;
    ChainOp &t = pt.ops[0] = make_op(EPI_AXPBY, 1.f, 0.f);
    set2(t.a, hh, hh); set2(t.a_lo, hl, hl); set2(t.b, 6, 6); set2(t.b_lo, 7, 7);
    set2(t.out16, 8, 8); set2(t.out16_lo, 9, 9);
    CHECK(run_chain(ctx, b, pt, nullptr, false, st));
    ChainProgram pa = one_shot(g1);
    pa.n_ops = 1;
    ChainOp &at = pa.ops[0] = make_op(EPI_AXPBY, 1.f, 0.f);
    set2(at.a, 6, 6); set2(at.a_lo, 7, 7); set2(at.b, 8, 8); set2(at.b_lo, 9, 9);
    at.use_div = 1; at.cout32 = 3;
    CHECK(run_chain(ctx, b, pa, b->d_scale, false, st));
    LAUNCH(ctx, launch_own_join(b, b->row_ptr, b->col_idx, b->h[6], b->h[7], b->u[2], st));
    b->lowdin = true;
    b->sinv_hi = b->sinv_lo = -1;
    b->sinv32_full = false;
    b->sinv_own_only = true;
    b->engine_simt = false;
    b->prepared = true;
    b->prepared_precision = precision;
    *gemms += inv_gemm_sum + 2 * b->count;
    return NOLSM_OK;
  }
  // S^-1 = Z^2 / s_S (Eq. 17); FP32 result -> u2, split copy -> (si_hi, si_lo).  The operands are the FP16
  // copies of Z the chain itself wrote last (parity_from_iters), so no conversion pass is needed.  When a
  // Newton refinement follows (it squares the error) plain FP16 operands are enough; otherwise split Z.
  const bool z_split = refine == 0;
  int si_hi, si_lo;           // where the split S^-1 lives
  {
    ChainProgram p1 = one_shot(g1);
    p1.n_ops = 1;
    p1.parity_from_iters = 1;
    ChainOp &o = p1.ops[0] = make_op(EPI_AXPBY, 1.f, 0.f);
    if (fp16) {               // Z16 in h2 / h3 (chain op z), Y16 buffers h0, h1 are free
      set2(o.a, 2, 3); set2(o.b, 2, 3);
      si_hi = 0; si_lo = 1;
      if (x0_direct) si_hi = 4;   // the E buffer: h0 will receive X0 while A0 is still an operand
    } else {                  // split Z in (h4,h5) / (h6,h7), split Y buffers h0..h3 are free
      set2(o.a, 4, 6); set2(o.b, 4, 6);
      if (z_split) { set2(o.a_lo, 5, 7); set2(o.b_lo, 5, 7); }
      si_hi = 2; si_lo = 3;
    }
    // with a refinement behind it S^-1 only continues as the split pair; its FP32 form is not needed
    o.use_div = 1; o.cout32 = refine > 0 ? -1 : 2; set2(o.out16, si_hi, si_hi);
    if (!fast_b) set2(o.out16_lo, si_lo, si_lo);
    CHECK(run_chain(ctx, b, p1, b->d_scale, false, st));
  }
  // split S (refinements) and split H (B = S^-1 H) come from the builder, in the last four halves
  const int ss_hi = b->n_half - 4, ss_lo = b->n_half - 3, hs_hi = b->n_half - 2, hs_lo = b->n_half - 1;
  // a pair of halves the iterations no longer need; FP16 mode: h3 (a Z buffer) and h5, which the sign iteration
  // (h0, h1, h2, h4) leaves alone, so that the split S^-1 of ONE refinement survives it (join_sinv)
  int fr_hi = fp16 ? 3 : 0, fr_lo = fp16 ? 5 : 1;
  if (refine > 0 && !b->s_split_built)           // batch built under another configuration
    LAUNCH(ctx, launch_scale_copy(b, S, nullptr, 0, nullptr, b->h[ss_hi], b->h[ss_lo], st));
  if (fast_b) {
    // A0: h0.  B0 = fp16(A0 H) -> h1 (whatever B0 is, the refinement only needs the SAME B0 in both places, so the
    // FP16 result is B0 and no lo part exists);  R = H - S B0 with S split, B0 exact -> h5;  B1 = B0 + A0 R -> u3.
    // Three launches: the plain products run on 256-row tiles, the half-split one on 128-row tiles.
    ChainProgram p5 = one_shot(g1);
    p5.n_ops = 1;
    ChainOp &b0 = p5.ops[0] = make_op(EPI_AXPBY, 1.f, 0.f);
    set2(b0.a, si_hi, si_hi); set2(b0.b, hs_hi, hs_hi); set2(b0.out16, 1, 1);
    CHECK(run_chain(ctx, b, p5, nullptr, false, st));
    ChainProgram p6 = one_shot(g1);
    p6.n_ops = 1;
    ChainOp &r = p6.ops[0] = make_op(EPI_AXPBY, -1.f, 1.f);
    set2(r.a, ss_hi, ss_hi); set2(r.a_lo, ss_lo, ss_lo); set2(r.b, 1, 1);
    set2(r.cin16, hs_hi, hs_hi); set2(r.cin16_lo, hs_lo, hs_lo); set2(r.out16, 5, 5);
    CHECK(run_chain(ctx, b, p6, nullptr, false, st));
    ChainProgram p7 = one_shot(g1);
    p7.n_ops = 1;
    ChainOp &b1 = p7.ops[0] = make_op(EPI_AXPBY, 1.f, 1.f);
    set2(b1.a, si_hi, si_hi); set2(b1.b, 5, 5); set2(b1.cin16, 1, 1);
    if (x0_direct) {
      // X0 = (B0 + A0 R - mu I)/s_j straight from the epilogue (hi -> h0, lo -> h2, where the sign iteration
      // expects its iterate), s_j from the norm bound of B0 - mu I, 1 % up for B1 - B0 (which is <= 2 r ~ 0.6 %
      // of B; the scale leaves 15 % to the edge of the convergence interval anyway, reading 5)
      LAUNCH(ctx, launch_norm_bound16(b, b->h[1], (float)*x0_mu, b->d_norm, st));
      LAUNCH(ctx, launch_x0_scale(b, b->d_norm, 1.01f, b->d_scale, st));
      b1.use_div = 2;
      b1.diag = -(float)*x0_mu;
      set2(b1.out16, 0, 0); set2(b1.out16_lo, 2, 2);
      CHECK(run_chain(ctx, b, p7, b->d_scale, false, st));
      b->x0_built = true;
      b->x0_mu = *x0_mu;
      b->b32_built = false;
    } else if (fp32_fast) {
      // B1 -> split pair (h6, h7); R2 = H - S B1 on full-split operands -> h5 (it is ~1e-4 |H|: FP16 holds it to
      // 5e-8); B2 = B1 + A0 R2 -> u3
      set2(b1.out16, 6, 6); set2(b1.out16_lo, 7, 7);
      CHECK(run_chain(ctx, b, p7, nullptr, false, st));
      ChainProgram p8 = one_shot(g1);
      p8.n_ops = 1;
      ChainOp &r2 = p8.ops[0] = make_op(EPI_AXPBY, -1.f, 1.f);
      set2(r2.a, ss_hi, ss_hi); set2(r2.a_lo, ss_lo, ss_lo); set2(r2.b, 6, 6); set2(r2.b_lo, 7, 7);
      set2(r2.cin16, hs_hi, hs_hi); set2(r2.cin16_lo, hs_lo, hs_lo); set2(r2.out16, 5, 5);
      CHECK(run_chain(ctx, b, p8, nullptr, false, st));
      ChainProgram p9 = one_shot(g1);
      p9.n_ops = 1;
      ChainOp &b2 = p9.ops[0] = make_op(EPI_AXPBY, 1.f, 1.f);
      set2(b2.a, si_hi, si_hi); set2(b2.b, 5, 5); set2(b2.cin16, 6, 6); set2(b2.cin16_lo, 7, 7);
      b2.cout32 = 3;
      CHECK(run_chain(ctx, b, p9, nullptr, false, st));
    } else {
      b1.cout32 = 3;
      CHECK(run_chain(ctx, b, p7, nullptr, false, st));
    }
    CHECK(ensure_thin(ctx, b, st));
    LAUNCH(ctx, launch_own_refine(b, b->row_ptr, b->col_idx, b->h[ss_hi], b->h[ss_lo], b->h[si_hi], b->d_thin, b->u[2],
                                  fp32_fast ? 2 : 1, st));
    b->sinv_hi = b->sinv_lo = -1;
    b->sinv32_full = false;
    b->sinv_own_only = true;
    b->engine_simt = false;
    b->prepared = true;
    b->prepared_precision = precision;
    *gemms += inv_gemm_sum;
    return NOLSM_OK;
  }
  b->sinv_own_only = false;
  for (int it = 0; it < refine; ++it) {
    // Newton refinement S^-1 <- S^-1 + S^-1 (I - S S^-1): the residual on split operands, the small
    // correction on plain FP16 operands (reading 11); the refined S^-1 leaves the epilogue as
    // FP32 master (u2) and as split copy in the free pair of halves.
    ChainProgram p2 = one_shot(g1);
    p2.n_ops = 2;
    ChainOp &r = p2.ops[0] = make_op(EPI_IDENT, 1.f, 0.f);
    set2(r.a, ss_hi, ss_hi); set2(r.a_lo, ss_lo, ss_lo); set2(r.b, si_hi, si_hi); set2(r.b_lo, si_lo, si_lo);
    set2(r.out16, 4, 4);
    ChainOp &c = p2.ops[1] = make_op(EPI_AXPBY, 1.f, 1.f);
    set2(c.a, si_hi, si_hi); set2(c.b, 4, 4); set2(c.cin16, si_hi, si_hi); set2(c.cin16_lo, si_lo, si_lo);
    set2(c.out16, fr_hi, fr_hi); set2(c.out16_lo, fr_lo, fr_lo);
    CHECK(run_chain(ctx, b, p2, nullptr, false, st));
    std::swap(si_hi, fr_hi); std::swap(si_lo, fr_lo);
  }
  // B = S^-1 H on split operands; result -> u3
  {
    ChainProgram p4 = one_shot(g1);
    p4.n_ops = 1;
    ChainOp &o = p4.ops[0] = make_op(EPI_AXPBY, 1.f, 0.f);
    set2(o.a, si_hi, si_hi); set2(o.a_lo, si_lo, si_lo); set2(o.b, hs_hi, hs_hi); set2(o.b_lo, hs_lo, hs_lo);
    o.cout32 = 3;
    CHECK(run_chain(ctx, b, p4, nullptr, false, st));
  }
  // a5 reads the six own columns of S^-1 only: they are joined to FP32 here, the rest on demand (join_sinv)
  b->sinv_hi = b->sinv_lo = -1;
  b->sinv32_full = true;
  if (refine > 0) {
    b->sinv_hi = si_hi; b->sinv_lo = si_lo;
    b->sinv32_full = false;
    if (fp16 && si_hi == 3 && b->sparse && b->grouped) {
      LAUNCH(ctx, launch_own_join_grouped(b, b->h[si_hi], b->h[si_lo], b->u[2], st));
    } else if (fp16 && si_hi == 3 && b->sparse && b->row_ptr) {
      LAUNCH(ctx, launch_own_join(b, b->row_ptr, b->col_idx, b->h[si_hi], b->h[si_lo], b->u[2], st));
    } else {   // the pair will be overwritten by the sign iteration: join all of it now
      CHECK(join_sinv(ctx, b, st));
      b->sinv_hi = b->sinv_lo = -1;
    }
  }
  b->engine_simt = false;
  b->prepared = true;
  b->prepared_precision = precision;
  *gemms += inv_gemm_sum;
  return NOLSM_OK;
}

// a3 (second part) + a4 on the tensor cores: X0 = (B - mu I)/s, then Eq. 9-10 in the correction form
// E = I - X_k^2,  X_{k+1} = X_k + 1/2 X_k E  (reading 12); the residual of the stop rule
// (reading 9) comes out of the first product's epilogue.  One kernel launch for all iterations.
static nolsm_status sign_batch_chain(nolsm_ctx *ctx, nolsm_batch *b, double mu, int precision, float tol,
                                     int max_iter, int fixed_iter, const float *scale_in, cudaStream_t st,
                                     bool timed, bool fold_last) {
  const bool fp16 = precision == NOLSM_FP16_FP32;
  float *Bm = b->u[3], *X32 = b->u[0];
  // the prepare stage of the whole path may have left X0 for this mu in place (prepare_batch_chain, x0_mu)
  const bool x0_ready = fp16 && b->x0_built && b->x0_mu == mu && !scale_in;
  b->x0_built = false;
  if (!x0_ready && !b->b32_built) { ctx->err = "this batch holds no B (its X0 was consumed)"; return NOLSM_EINVAL; }
  if (!scale_in && !x0_ready) LAUNCH(ctx, launch_norm_bound(b, Bm, (float)mu, false, b->d_norm, st));
  ChainProgram pg;
  memset(&pg, 0, sizeof(pg));
  pg.n_ops = 2;
  pg.max_iter = max_iter;
  pg.fixed_iter = fixed_iter > 0 ? fixed_iter : 0;
  pg.tol = tol;
  // fold_last: stop right after the E_k that passes the test; the caller applies X_{k+1} = X_k + 1/2 X_k E_k
  // only to the own columns of S^-1 (k_thin_mma<kLastHalf>), instead of forming it with an n^3 product
  const bool order3 = fp16 && (ctx->cfg.flags & NOLSM_FLAG_ORDER3) != 0;
  bool rescale = false;
  b->sign_iter0 = 0;
  if (order3) fold_last = false;   // the folded update is Eq. 9's
  pg.stop_early = fold_last ? 1 : 0;
  b->x_pending = fold_last;
  b->x_pending_split = fold_last && !fp16;
  b->sign_ops = order3 ? 3 : 2;
  ChainOp &e = pg.ops[0] = make_op(EPI_IDENT, 1.f, 0.f);
  ChainOp &x = pg.ops[1] = make_op(EPI_AXPBY, 0.5f, 1.f);
  e.resid = 1;
  b->x_split = true;
  b->x32_valid = false;
  if (fp16) {
    // Master iterate as hi + lo * 2^-11 (22 bits, reading 12): hi IS the FP16 operand X16 (h0/h1,
    // ping-pong), lo lives in h2 and is updated in place by the thread that owns the element; E16: h4.
    // Per element and iteration the epilogues write 6 bytes (E, hi, lo) instead of 8 (E, FP32 master, FP16 copy).
    if (!x0_ready)
      LAUNCH(ctx, launch_make_x0(b, Bm, (float)mu, b->d_norm, scale_in, nullptr, b->h[0], b->h[2], b->d_scale, st));
    pg.group = group_size(ctx, b, 6);
    set2(e.a, 0, 1); set2(e.b, 0, 1); set2(e.out16, 4, 4);
    set2(x.a, 0, 1); set2(x.b, 4, 4); set2(x.cin16, 0, 1); set2(x.cin16_lo, 2, 2);
    set2(x.out16, 1, 0); set2(x.out16_lo, 2, 2); x.lo_stream = 1;
    // rescaled first iteration (reading 5): ||X0^2||_1 from E_0's epilogue bounds rho(X0) tighter than the O(n^2)
    // norm bound X0 was scaled with; iteration 0 is applied to a X0 with a = 1.7 / sqrt(||X0^2||_1) >= 1
    rescale = !order3 && !scale_in && ctx->cfg.gap_hint <= 0.f && pg.fixed_iter <= 0 && max_iter > 1 &&
              (ctx->cfg.flags & NOLSM_FLAG_NO_RESCALE) == 0;
    if (order3) {
      // X <- X (I + 1/2 E + 3/8 E^2) = X + X G,  G = 1/2 E + 3/8 E E  (refs [51],[52]); G in a half the
      // iterations do not use: the builder's split copy of S (sparse batches, free after the prepare stage) or h5
      const int gbuf = b->sparse ? b->n_half - 4 : 5;
      pg.n_ops = 3;
      pg.ops[2] = x;
      ChainOp &g = pg.ops[1] = make_op(EPI_AXPBY, 0.375f, 0.5f);
      set2(g.a, 4, 4); set2(g.b, 4, 4); set2(g.cin16, 4, 4); set2(g.out16, gbuf, gbuf);
      ChainOp &x3 = pg.ops[2];
      x3.alpha = 1.f;
      set2(x3.b, gbuf, gbuf);
    }
  } else {
    // split operands: X (h0,h1)/(h2,h3), E (h4,h5)
    // the master iterate is the split operand pair itself (no FP32 copy): X (h0,h1) / (h2,h3) ping-pong
    LAUNCH(ctx, launch_make_x0(b, Bm, (float)mu, b->d_norm, scale_in, nullptr, b->h[0], b->h[1], b->d_scale, st));
    pg.group = group_size(ctx, b, 12);
    set2(e.a, 0, 2); set2(e.a_lo, 1, 3); set2(e.b, 0, 2); set2(e.b_lo, 1, 3);
    set2(e.out16, 4, 4); set2(e.out16_lo, 5, 5);
    set2(x.a, 0, 2); set2(x.a_lo, 1, 3); set2(x.b, 4, 4); set2(x.b_lo, 5, 5);
    set2(x.cin16, 0, 2); set2(x.cin16_lo, 1, 3);
    set2(x.out16, 2, 0); set2(x.out16_lo, 3, 1);
    rescale = !scale_in && ctx->cfg.gap_hint <= 0.f && pg.fixed_iter <= 0 && max_iter > 1 &&
              (ctx->cfg.flags & NOLSM_FLAG_NO_RESCALE) == 0;
  }
  if (ctx->cfg.gap_hint > 0.f && !scale_in && pg.fixed_iter <= 0) {   // scaled start
    LAUNCH(ctx, launch_alpha_schedule(b, b->d_scale, ctx->cfg.gap_hint, b->d_alpha, st));
    pg.use_alpha_tab = 1;
  }
  if (timed) NOLSM_CUDA(ctx, cudaEventRecord(ctx->tev[0], st));
  if (rescale) {
    // Iteration 0 in a launch of its own (the kernel instantiation with the column norms and the per-matrix scale;
    // the other iterations keep the plain one): E_0 gathers ||X0^2||_1, the X update applies a (ChainOp::colnorm 2)
    ChainProgram p0 = one_shot(pg.group);
    p0.n_ops = 2;
    p0.tol = tol;
    p0.ops[0] = e;
    p0.ops[1] = x;
    p0.ops[0].colnorm = p0.ops[1].colnorm = 2;
    p0.rescale_target = 1.7f;   // < sqrt 3 = 1.732; measured: 1.6 leaves half of the n ~ 1489 submatrices one iteration short
    CHECK(run_chain(ctx, b, p0, nullptr, false, st));
    // the adaptive launch starts at iteration 1: its tables are indexed by the parity of ITS iteration count
    auto flip = [](int32_t (&d)[2]) { std::swap(d[0], d[1]); };
    for (ChainOp *o : {&e, &x}) {
      flip(o->a); flip(o->b); flip(o->a_lo); flip(o->b_lo); flip(o->out16); flip(o->out16_lo);
      flip(o->cin16); flip(o->cin16_lo);
    }
    pg.max_iter = max_iter - 1;
    b->sign_iter0 = 1;
  }
  CHECK(run_chain(ctx, b, pg, nullptr, true, st));
  if (timed) NOLSM_CUDA(ctx, cudaEventRecord(ctx->tev[1], st));
  NOLSM_CUDA(ctx, cudaMemcpyAsync(b->d_sched + 5, b->d_sched + 2, sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
  return NOLSM_OK;
}

// ---- debugging path: every product on the FP32 SIMT kernel (NOLSM_FLAG_SIMT_ONLY) ----
struct Engine {
  nolsm_ctx *ctx;
  nolsm_batch *b;
  cudaStream_t st;
  int64_t gemms = 0;

  GemmParams base_params() const {
    GemmParams p;
    memset(&p, 0, sizeof(p));
    p.tiles = b->d_tiles_simt;
    p.n_tiles = b->n_tiles_simt;
    p.dims = b->d_dims;
    p.ld = b->ld;
    p.slab = (int64_t)b->ld * b->ld;
    p.alpha = 1.f;
    return p;
  }
  nolsm_status simt(int mode, float alpha, float beta, const float *alpha_div, const float *a, const float *bb,
                    const float *cin, float *cout, float *resid2, const int32_t *state, int iter) {
    GemmParams p = base_params();
    p.mode = mode; p.alpha = alpha; p.beta = beta; p.alpha_div = alpha_div;
    p.a32 = a; p.b32 = bb; p.cin32 = cin; p.cout32 = cout; p.resid2 = resid2;
    p.state = state; p.iter = iter;
    LAUNCH(ctx, launch_gemm_simt(p, st));
    gemms++;
    return NOLSM_OK;
  }
  float *resid_slot(int iter) const { return b->d_resid2 + (size_t)(iter % NOLSM_MAX_RESID_SLOTS) * b->count; }
  nolsm_status zero_resid(int iter) {
    NOLSM_CUDA(ctx, cudaMemsetAsync(resid_slot(iter), 0, sizeof(float) * b->count, st));
    return NOLSM_OK;
  }
  nolsm_status control(int phase, int iter, float tol, int max_iter, int fixed_iter, bool lockstep) {
    LAUNCH(ctx, launch_control(b, phase | (lockstep ? 16 : 0), iter, tol, max_iter, fixed_iter, st));
    return NOLSM_OK;
  }
  // Lagged host check: after iteration k the active count is copied out; before launching iteration
  // k+2 the host looks at it.
  nolsm_status post_active(int k) {
    NOLSM_CUDA(ctx, cudaMemcpyAsync(&ctx->h_active[k], &b->d_active[k], sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    NOLSM_CUDA(ctx, cudaEventRecord(ctx->ev[k & 3], st));
    return NOLSM_OK;
  }
  nolsm_status finished(int k, bool *done) {
    NOLSM_CUDA(ctx, cudaEventSynchronize(ctx->ev[k & 3]));
    *done = ctx->h_active[k] == 0;
    return NOLSM_OK;
  }
};

template <typename Body>
static nolsm_status iterate(Engine &E, int max_iter, int fixed_iter, int *executed, Body body) {
  const int limit = fixed_iter > 0 ? std::min(fixed_iter, max_iter) : max_iter;
  int k = 0;
  for (; k < limit; ++k) {
    if (fixed_iter <= 0 && k >= 2) {
      bool done = false;
      CHECK(E.finished(k - 2, &done));
      if (done) break;
    }
    CHECK(body(k));
    CHECK(E.post_active(k));
  }
  NOLSM_CUDA(E.ctx, cudaStreamSynchronize(E.st));
  *executed = k;
  for (int i = 0; i < k; ++i)
    if (E.ctx->h_active[i] == 0) { *executed = i + 1; break; }
  return NOLSM_OK;
}

static nolsm_status prepare_batch_simt(nolsm_ctx *ctx, nolsm_batch *b, cudaStream_t st, nolsm_sign_stats *stats,
                                       int64_t *gemms) {
  Engine E{ctx, b, st};
  const float inv_tol = ctx->cfg.inv_tol > 0.f ? ctx->cfg.inv_tol : 1e-5f;
  const int max_it = ctx->cfg.inv_max_iter;
  float *S = b->u[0], *H = b->u[1];
  LAUNCH(ctx, launch_norm_bound(b, S, 0.f, true, b->d_norm, st));
  CHECK(E.control(0, 0, 0.f, 0, 0, false));
  int executed = 0;
  float *Y[2] = {b->u[2], b->u[5]}, *Z[2] = {b->u[3], b->u[6]}, *Em = b->u[4];
  LAUNCH(ctx, launch_init_inverse(b, S, b->d_norm, Y[0], Z[0], nullptr, nullptr, nullptr, nullptr, b->d_scale, st));
  CHECK(iterate(E, max_it, 0, &executed, [&](int k) -> nolsm_status {
    const int cur = k & 1, nxt = cur ^ 1;
    CHECK(E.zero_resid(k));
    CHECK(E.simt(EPI_IDENT, 1.f, 0.f, nullptr, Z[cur], Y[cur], nullptr, Em, E.resid_slot(k), b->d_state, k));
    CHECK(E.control(1, k, inv_tol, max_it, 0, true));
    CHECK(E.simt(EPI_AXPBY, 0.5f, 1.f, nullptr, Y[cur], Em, Y[cur], Y[nxt], nullptr, b->d_state, k));
    CHECK(E.simt(EPI_AXPBY, 0.5f, 1.f, nullptr, Em, Z[cur], Z[cur], Z[nxt], nullptr, b->d_state, k));
    return NOLSM_OK;
  }));
  float *Zf = Z[executed & 1];
  CHECK(E.simt(EPI_AXPBY, 1.f, 0.f, b->d_scale, Zf, Zf, nullptr, b->u[4], nullptr, nullptr, 0));
  CHECK(E.simt(EPI_AXPBY, 1.f, 0.f, nullptr, b->u[4], H, nullptr, b->u[2], nullptr, nullptr, 0));
  b->engine_simt = true;
  b->prepared = true;
  b->prepared_precision = NOLSM_FP32;
  if (stats) {
    stats->inv_iter_max = executed;
    stats->flops_prepare = 2.0 * b->sum_n3 * (double)E.gemms;
    std::vector<float> res(b->count);
    NOLSM_CUDA(ctx, cudaMemcpyAsync(res.data(), b->d_lastres, sizeof(float) * b->count, cudaMemcpyDeviceToHost, st));
    NOLSM_CUDA(ctx, cudaStreamSynchronize(st));
    for (float r : res)
      if (!(r <= stats->inv_worst_residual)) stats->inv_worst_residual = r;
  }
  *gemms += E.gemms * b->count;
  return NOLSM_OK;
}

static nolsm_status sign_batch_simt(nolsm_ctx *ctx, nolsm_batch *b, double mu, float tol, int max_iter,
                                    int fixed_iter, const float *scale_in, cudaStream_t st) {
  Engine E{ctx, b, st};
  float *Bm = b->u[2];
  if (!scale_in) LAUNCH(ctx, launch_norm_bound(b, Bm, (float)mu, false, b->d_norm, st));
  CHECK(E.control(0, 0, 0.f, 0, 0, false));
  int executed = 0;
  float *X[2] = {b->u[0], b->u[3]}, *Em = b->u[5];
  LAUNCH(ctx, launch_make_x0(b, Bm, (float)mu, b->d_norm, scale_in, X[0], nullptr, nullptr, b->d_scale, st));
  CHECK(iterate(E, max_iter, fixed_iter, &executed, [&](int k) -> nolsm_status {
    const int cur = k & 1, nxt = cur ^ 1;
    CHECK(E.zero_resid(k));
    CHECK(E.simt(EPI_IDENT, 1.f, 0.f, nullptr, X[cur], X[cur], nullptr, Em, E.resid_slot(k), b->d_state, k));
    CHECK(E.control(1, k, tol, max_iter, fixed_iter, true));
    CHECK(E.simt(EPI_AXPBY, 0.5f, 1.f, nullptr, X[cur], Em, X[cur], X[nxt], nullptr, b->d_state, k));
    return NOLSM_OK;
  }));
  b->x_parity = executed & 1;
  return NOLSM_OK;
}

static nolsm_status prepare_batch(nolsm_ctx *ctx, nolsm_batch *b, int precision, cudaStream_t st,
                                  nolsm_sign_stats *stats, int64_t *gemms, bool own_only = false,
                                  const double *x0_mu = nullptr) {
  b->sinv_own_only = false;
  if (use_simt(ctx)) return prepare_batch_simt(ctx, b, st, stats, gemms);
  return prepare_batch_chain(ctx, b, precision, st, stats, gemms, own_only, x0_mu);
}

// timed: records ctx->tev[0..1] around the chain kernel; read with chain_ms() after a synchronise
static nolsm_status sign_batch(nolsm_ctx *ctx, nolsm_batch *b, double mu, int precision, float tol, int max_iter,
                               int fixed_iter, const float *scale_in, cudaStream_t st, bool timed,
                               bool fold_last = false) {
  b->x_pending = false;
  b->x_split = false;
  b->x32_valid = true;
  if (b->engine_simt) return sign_batch_simt(ctx, b, mu, tol, max_iter, fixed_iter, scale_in, st);
  return sign_batch_chain(ctx, b, mu, precision, tol, max_iter, fixed_iter, scale_in, st, timed, fold_last);
}

// SM cycles of the last chain kernel of the batch (max over its CTAs), in millions; synchronises
static float chain_mcycles(nolsm_ctx *ctx, const nolsm_batch *b, cudaStream_t st) {
  int32_t kc = 0;
  if (b->engine_simt || b->count == 0) return 0.f;
  if (cudaMemcpyAsync(&kc, b->d_sched + 3, sizeof(int32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess) { cudaGetLastError(); return 0.f; }
  return (float)kc * (1024.f / 1e6f);
}

static float chain_ms(nolsm_ctx *ctx, const nolsm_batch *b) {
  float ms = 0.f;
  if (b->engine_simt || b->count == 0) return 0.f;
  if (cudaEventElapsedTime(&ms, ctx->tev[0], ctx->tev[1]) != cudaSuccess) { cudaGetLastError(); return 0.f; }
  return ms;
}

static float *sinv_ptr(const nolsm_batch *b) { return b->engine_simt ? b->u[4] : b->u[2]; }
static float *bmat_ptr(const nolsm_batch *b) { return b->engine_simt ? b->u[2] : b->u[3]; }
static float *x_ptr(const nolsm_batch *b) { return (b->engine_simt && b->x_parity) ? b->u[3] : b->u[0]; }
static XRef x_ref(const nolsm_batch *b) {
  if (b->x_split && !b->engine_simt) {
    if (b->prepared_precision == NOLSM_FP16_FP32)   // (buffer by the parity of d_iters, which may count from iteration 1)
      return (b->sign_iter0 & 1) ? XRef{nullptr, b->h[1], b->h[0], b->h[2], b->h[2]}
                                 : XRef{nullptr, b->h[0], b->h[1], b->h[2], b->h[2]};
    return (b->sign_iter0 & 1) ? XRef{nullptr, b->h[2], b->h[0], b->h[3], b->h[1]}
                               : XRef{nullptr, b->h[0], b->h[2], b->h[1], b->h[3]};
  }
  return XRef{x_ptr(b), nullptr, nullptr, nullptr, nullptr};
}
// full FP32 S^-1 in u2 (the prepare stage leaves only its own columns there), for the consumers that read all of it
// scratch of the thin (n x 6) products: 2 * count * 6 * ld floats
static nolsm_status ensure_thin(nolsm_ctx *ctx, nolsm_batch *b, cudaStream_t st) {
  const size_t need = (size_t)2 * b->count * NOLSM_BS * b->ld;
  if (need <= b->thin_cap) return NOLSM_OK;
  cudaStreamSynchronize(st);
  cudaFree(b->d_thin);
  b->d_thin = nullptr;
  b->thin_cap = 0;
  if (need && cudaMalloc(&b->d_thin, need * sizeof(float)) != cudaSuccess) {
    cudaGetLastError();
    ctx->err = "cudaMalloc of the thin-product scratch failed";
    return NOLSM_ENOMEM;
  }
  b->thin_cap = need;
  return NOLSM_OK;
}

static nolsm_status join_sinv(nolsm_ctx *ctx, nolsm_batch *b, cudaStream_t st) {
  if (b->sinv_own_only) { ctx->err = "this batch holds the own columns of S^-1 only"; return NOLSM_EINVAL; }
  if (b->engine_simt || b->sinv32_full || b->sinv_hi < 0) return NOLSM_OK;
  LAUNCH(ctx, launch_join_split(b, XRef{nullptr, b->h[b->sinv_hi], b->h[b->sinv_hi], b->h[b->sinv_lo], b->h[b->sinv_lo]},
                                b->u[2], st));
  b->sinv32_full = true;
  return NOLSM_OK;
}
// FP32 copy of a split sign iterate in u0, for the consumers that read X as FP32
static nolsm_status join_x(nolsm_ctx *ctx, nolsm_batch *b, cudaStream_t st) {
  if (!b->x_split || b->engine_simt || b->x32_valid) return NOLSM_OK;
  LAUNCH(ctx, launch_join_split(b, x_ref(b), b->u[0], st));
  b->x32_valid = true;
  return NOLSM_OK;
}

// Collect per-submatrix iteration counts and residuals (synchronises).
static nolsm_status collect_stats(nolsm_ctx *ctx, nolsm_batch *b, float tol, int fixed_iter, cudaStream_t st,
                                  nolsm_sign_stats *s) {
  std::vector<int32_t> it(b->count);
  std::vector<float> res(b->count);
  NOLSM_CUDA(ctx, cudaMemcpyAsync(it.data(), b->d_iters, sizeof(int32_t) * b->count, cudaMemcpyDeviceToHost, st));
  NOLSM_CUDA(ctx, cudaMemcpyAsync(res.data(), b->d_lastres, sizeof(float) * b->count, cudaMemcpyDeviceToHost, st));
  NOLSM_CUDA(ctx, cudaStreamSynchronize(st));
  s->n_sub = b->count;
  s->iter_min = b->count ? 1 << 30 : 0;
  s->iter_max = 0;
  s->iter_sum = 0;
  s->n_unconverged = 0;
  s->worst_residual = 0.f;
  s->flops_sign = s->flops_sign_padded = 0.0;
  for (int m = 0; m < b->count; ++m) {
    // a folded last iteration: the chain counted the iterations it carried out in full and ran one product more
    const int extra = b->x_pending ? 1 : 0;
    const double n3 = (double)b->n_host[m] * b->n_host[m] * b->n_host[m];
    const double P3 = (double)round_up(b->n_host[m], NOLSM_TILE_M) * round_up(b->n_host[m], 64) * round_up(b->n_host[m], 64);
    s->flops_sign -= extra * 2.0 * n3;          // (2 it + 1) products instead of 2 (it + 1)
    s->flops_sign_padded -= extra * 2.0 * P3;
    it[m] += extra + b->sign_iter0;
    s->iter_min = std::min(s->iter_min, it[m]);
    s->iter_max = std::max(s->iter_max, it[m]);
    s->iter_sum += it[m];
    if (!(res[m] < tol) && fixed_iter <= 0) s->n_unconverged++;
    if (!(res[m] <= s->worst_residual)) s->worst_residual = res[m];
    const double n = b->n_host[m], P = round_up(b->n_host[m], NOLSM_TILE_M), Pn = round_up(b->n_host[m], 64);
    s->flops_sign += 2.0 * it[m] * (double)b->sign_ops * n * n * n;
    s->flops_sign_padded += 2.0 * it[m] * (double)b->sign_ops * P * Pn * Pn;
  }
  return NOLSM_OK;
}

static void resolve_sign_args(const nolsm_ctx *ctx, int precision, float *tol, int *max_iter, int *fixed_iter) {
  if (*tol <= 0.f) *tol = ctx->cfg.tol > 0.f ? ctx->cfg.tol : (precision == NOLSM_FP16_FP32 ? 1e-2f : 1e-5f);
  if (*max_iter <= 0) *max_iter = ctx->cfg.max_iter;
  if (*max_iter > NOLSM_MAX_RESID_SLOTS) *max_iter = NOLSM_MAX_RESID_SLOTS;
  if (*fixed_iter < 0) *fixed_iter = ctx->cfg.fixed_iter;
  if (*fixed_iter > *max_iter) *fixed_iter = *max_iter;
}

extern "C" nolsm_status nolsm_sign_batched(nolsm_ctx *ctx, nolsm_batch *batch, double mu, int32_t precision,
                                           float tol, int32_t max_iter, int32_t fixed_iter,
                                           nolsm_sign_stats *stats, void *stream) {
  if (!ctx || !batch) return NOLSM_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const int prec = effective_precision(ctx, precision);
  if (prec != NOLSM_FP16_FP32 && prec != NOLSM_FP32) { ctx->err = "bad precision"; return NOLSM_EINVAL; }
  resolve_sign_args(ctx, prec, &tol, &max_iter, &fixed_iter);
  if (stats) memset(stats, 0, sizeof(*stats));
  int64_t gemms = 0;
  if (batch->n_unit < units_for(prec)) {
    ctx->err = "batch was built for another precision (create the context with the precision you run)";
    return NOLSM_EINVAL;
  }
  if (!batch->prepared || batch->prepared_precision != prec) {
    if (!batch->sparse) { ctx->err = "dense batch is not prepared"; return NOLSM_EINVAL; }
    if (batch->prepared) { ctx->err = "batch was prepared in another precision; gather it again"; return NOLSM_EINVAL; }
    CHECK(prepare_batch(ctx, batch, prec, st, stats, &gemms));
  }
  CHECK(sign_batch(ctx, batch, mu, prec, tol, max_iter, fixed_iter, nullptr, st, stats != nullptr));
  int32_t bad[2] = {0, 0};   // the status is a scalar that must reach the host: this call synchronises here
  if (!batch->engine_simt) {
    NOLSM_CUDA(ctx, cudaMemcpyAsync(bad, batch->d_sched + 4, sizeof(bad), cudaMemcpyDeviceToHost, st));
    NOLSM_CUDA(ctx, cudaStreamSynchronize(st));
  }
  if (stats) {
    const int inv_it = stats->inv_iter_max;
    const float inv_res = stats->inv_worst_residual;
    const double fp = stats->flops_prepare;
    CHECK(collect_stats(ctx, batch, tol, fixed_iter, st, stats));
    stats->inv_iter_max = inv_it;
    stats->inv_worst_residual = inv_res;
    stats->flops_prepare = fp;
    stats->gemms = gemms + batch->sign_ops * stats->iter_sum;
    stats->ms_chain = chain_ms(ctx, batch);
    stats->chain_mcycles = chain_mcycles(ctx, batch, st);
    if (!batch->engine_simt) stats->n_unconverged = bad[1];
  }
  if (bad[0] > 0) {
    ctx->err = std::to_string(bad[0]) + " submatrices: Eq. 15-17 did not reach inv_tol within inv_max_iter (S_j not SPD?)";
    return NOLSM_ENOTSPD;
  }
  if (bad[1] > 0 && fixed_iter <= 0) {
    ctx->err = std::to_string(bad[1]) + " submatrices: the sign iteration hit max_iter";
    return NOLSM_ENOCONV;
  }
  return NOLSM_OK;
}

// ------------------------------------------------------------------------------------------------
// a5 - a7
// ------------------------------------------------------------------------------------------------
extern "C" nolsm_status nolsm_scatter_density(nolsm_ctx *ctx, const nolsm_batch *batch, const nolsm_bsr *S,
                                              nolsm_bsr *D, double *ne_partial, double *q_mol, double *ne_diag,
                                              void *stream) {
  if (!ctx || !batch || !ne_partial) return NOLSM_EINVAL;
  CHECK(check_bsr(ctx, S, "S"));
  CHECK(check_bsr(ctx, D, "D"));
  if (!batch->sparse || !batch->prepared) { ctx->err = "batch has no sign iterate (call nolsm_sign_batched first)"; return NOLSM_EINVAL; }
  if (D->n_mol != S->n_mol || D->row_ptr != S->row_ptr || D->col_idx != S->col_idx) {
    ctx->err = "D must share the pattern of S";
    return NOLSM_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)stream;
  if (batch->grouped) {   // combined submatrices: several owners per submatrix
    if (batch->x_pending || batch->engine_simt) { ctx->err = "combined submatrices need the finished tensor-core iterate"; return NOLSM_EINVAL; }
    LAUNCH(ctx, launch_density_grouped(batch, x_ref(batch), sinv_ptr(batch), S->row_ptr, S->col_idx, D->val, st));
    LAUNCH(ctx, launch_trace(batch, S->row_ptr, S->col_idx, D->val, S->val, ne_partial, q_mol, st));
    return NOLSM_OK;
  }
  float *u_thin = nullptr;
  if (batch->x_pending) {
    nolsm_batch *bm = const_cast<nolsm_batch *>(batch);
    CHECK(ensure_thin(ctx, bm, st));   // same scratch as the energy products
    u_thin = bm->d_thin;
  }
  if (batch->lowdin) {
    // Loewdin form: U = 1/2 (W - X~ W) with W = Z[:, own] (u2), then D[:, own] = Z U / s_S
    nolsm_batch *bm = const_cast<nolsm_batch *>(batch);
    CHECK(ensure_thin(ctx, bm, st));
    float *u_out = bm->d_thin + (size_t)batch->count * NOLSM_BS * batch->ld;   // second half of the scratch
    ctx->launches += 1;
    if (launch_density_split(batch, x_ref(batch), sinv_ptr(batch), S->row_ptr, S->col_idx, nullptr, nullptr, batch->h[4],
                             batch->x_pending_split ? batch->h[5] : nullptr, u_thin, st, u_out) != cudaSuccess) {
      cudaGetLastError(); ctx->err = "density columns (Loewdin form): launch failed"; return NOLSM_ECUDA;
    }
    LAUNCH(ctx, launch_scaled_out(batch, S->row_ptr, S->col_idx, batch->h[6], batch->h[7], u_out, batch->d_scale_s,
                                  D->val, st));
    LAUNCH(ctx, launch_trace(batch, S->row_ptr, S->col_idx, D->val, S->val, ne_partial, q_mol, st));
    return NOLSM_OK;
  }
  LAUNCH(ctx, launch_density(batch, x_ref(batch), sinv_ptr(batch), S->row_ptr, S->col_idx, D->val,
                             ne_diag, batch->h[4], batch->x_pending_split ? batch->h[5] : nullptr, u_thin, st));
  LAUNCH(ctx, launch_trace(batch, S->row_ptr, S->col_idx, D->val, S->val, ne_partial, q_mol, st));
  return NOLSM_OK;
}

// Eq. 7/11 and Eq. 8/13 for the molecules of a batch
extern "C" nolsm_status nolsm_scatter_energy(nolsm_ctx *ctx, nolsm_batch *batch, const nolsm_bsr *H,
                                             const nolsm_bsr *D, nolsm_bsr *W, double *e_partial, void *stream) {
  if (!ctx || !batch) return NOLSM_EINVAL;
  CHECK(check_bsr(ctx, H, "H"));
  if (!batch->sparse || !batch->prepared) { ctx->err = "batch has no sign iterate (call nolsm_sign_batched first)"; return NOLSM_EINVAL; }
  if (batch->x_pending) { ctx->err = "internal: the energy products need the finished sign iterate"; return NOLSM_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  if (W) {
    CHECK(check_bsr(ctx, W, "W"));
    if (W->n_mol != H->n_mol || W->row_ptr != H->row_ptr || W->col_idx != H->col_idx) {
      ctx->err = "W must share the pattern of H";
      return NOLSM_EINVAL;
    }
    const size_t need = (size_t)2 * batch->count * NOLSM_BS * batch->ld;
    if (need > batch->thin_cap) {
      cudaStreamSynchronize(st);
      cudaFree(batch->d_thin);
      batch->d_thin = nullptr;
      batch->thin_cap = 0;
      if (need && cudaMalloc(&batch->d_thin, need * sizeof(float)) != cudaSuccess) {
        cudaGetLastError(); ctx->err = "cudaMalloc of the thin-product scratch failed"; return NOLSM_ENOMEM;
      }
      batch->thin_cap = need;
    }
    CHECK(join_x(ctx, batch, st));
    CHECK(join_sinv(ctx, batch, st));
    cudaError_t e = launch_energy_weighted(batch, x_ptr(batch), sinv_ptr(batch), batch->u[1], H->row_ptr, H->col_idx,
                                           batch->d_thin, W->val, st);
    ctx->launches += 4;
    if (e != cudaSuccess) { ctx->err = std::string("energy-weighted density: ") + cudaGetErrorString(e); return NOLSM_ECUDA; }
  }
  if (e_partial) {
    CHECK(check_bsr(ctx, D, "D"));
    if (D->n_mol != H->n_mol || D->row_ptr != H->row_ptr || D->col_idx != H->col_idx) {
      ctx->err = "D must share the pattern of H";
      return NOLSM_EINVAL;
    }
    LAUNCH(ctx, launch_energy(batch, H->row_ptr, D->val, H->val, e_partial, st));
  }
  return NOLSM_OK;
}

// ------------------------------------------------------------------------------------------------
// Whole path with batching and bisection
// ------------------------------------------------------------------------------------------------
extern "C" nolsm_status nolsm_solve_mu(nolsm_ctx *ctx, const nolsm_bsr *H, const nolsm_bsr *S, double n_electrons,
                                       double mu_lo, double mu_hi, double tol_ne_per_mol, int32_t max_steps,
                                       int32_t precision, nolsm_bsr *D, double *mu_out, double *ne_out,
                                       double *q_mol, nolsm_solve_stats *stats, void *stream) {
  if (!ctx || !mu_out || !ne_out) return NOLSM_EINVAL;
  CHECK(check_bsr(ctx, H, "H"));
  CHECK(check_bsr(ctx, S, "S"));
  CHECK(check_bsr(ctx, D, "D"));
  if (!(mu_lo < mu_hi) || max_steps <= 0) { ctx->err = "need mu_lo < mu_hi and max_steps > 0"; return NOLSM_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const int prec = effective_precision(ctx, precision);
  if ((ctx->cfg.flags & NOLSM_FLAG_LOWDIN) != 0 &&
      (prec == NOLSM_FP16_FP32 || ctx->eval_energy || use_simt(ctx) || !ctx->umma_ok || ctx->has_model)) {
    ctx->err = "NOLSM_FLAG_LOWDIN: FP32 mode of nolsm_solve_mu only (it needs S^-1/2 at FP32 quality; no energy "
               "products, no generated elements)";
    return NOLSM_EINVAL;
  }
  float tol = 0.f;
  int max_iter = 0, fixed_iter = -1;
  resolve_sign_args(ctx, prec, &tol, &max_iter, &fixed_iter);
  const int n_mol = H->n_mol;
  if (stats) memset(stats, 0, sizeof(*stats));

  // batching plan from the neighbour counts
  std::vector<int32_t> dims;
  if (n_mol > 0) CHECK(read_dims(ctx, H->row_ptr, 0, n_mol, dims, st));
  struct Range { int begin, count; size_t bytes; };
  std::vector<Range> plan;
  const int units = units_for(prec);
  auto make_plan = [&](size_t budget, int max_count) -> bool {
    plan.clear();
    int i = 0;
    while (i < n_mol) {
      int max_n = 0, cnt = 0;
      while (i + cnt < n_mol && cnt < max_count) {
        const int mn = std::max(max_n, dims[i + cnt]);
        if (dense_bytes(cnt + 1, round_up(mn, NOLSM_PAD), units) > budget) break;
        max_n = mn;
        cnt++;
      }
      if (cnt == 0) return false;
      plan.push_back(Range{i, cnt, dense_bytes(cnt, round_up(max_n, NOLSM_PAD), units)});
      i += cnt;
    }
    return true;
  };
  const size_t ws = (size_t)ctx->cfg.workspace_bytes;
  const int max_count = 4096;
  bool resident = false;
  if (!make_plan(ws, max_count)) { ctx->err = "workspace_bytes cannot hold one submatrix"; return NOLSM_ENOMEM; }
  {
    size_t total = 0;
    for (const Range &r : plan) total += r.bytes;
    resident = total <= ws && plan.size() <= 64;
  }
  // The context's own slots are re-planned on every call: release those the plan does not use and those whose
  // workspace is far larger than the plan needs (a streaming call leaves one of the full workspace size behind),
  // so that the accounting against workspace_bytes is about what this call holds.
  {
    size_t user = 0;
    for (int i = 0; i < kUserSlots && i < (int)ctx->slots.size(); ++i)
      if (ctx->slots[i]) user += ctx->slots[i]->base_bytes;
    size_t total = 0;
    for (const Range &r : plan) total += r.bytes;
    resident = resident && total + user <= ws;
    for (int i = kOwnSlot; i < kOwnDense && i < (int)ctx->slots.size(); ++i) {
      nolsm_batch *ob = ctx->slots[i];
      if (!ob) continue;
      const int bi = i - kOwnSlot;
      const bool used = resident ? bi < (int)plan.size() : bi == 0;
      const size_t want = used ? (resident ? plan[bi].bytes : plan[0].bytes) : 0;
      if (!used || ob->base_bytes > want + want / 2 + ((size_t)64 << 20)) {
        cudaStreamSynchronize(st);
        free_batch(ob);
        ctx->slots[i] = nullptr;
      }
    }
  }
  std::vector<nolsm_batch *> live(plan.size(), nullptr);

  // Operator cache (nolsm_config.cache_bytes): streamed batches lose S^-1 and B between mu steps; keeping
  // B_j (FP32, padded slab) and the own columns of S_j^-1 lets steps 2.. start at the sign iteration.
  float *cache = nullptr;
  std::vector<size_t> cache_off(plan.size() + 1, 0), cache_sq(plan.size(), 0);
  if (!resident && max_steps > 1 && ctx->cfg.cache_bytes >= 0 && !use_simt(ctx) && ctx->umma_ok &&
      (ctx->cfg.flags & NOLSM_FLAG_LOWDIN) == 0) {   // (the Loewdin form keeps Z in the workspace: no cache)
    for (size_t bi = 0; bi < plan.size(); ++bi) {
      int max_n = 0;
      size_t sq = 0;     // B_j packed to its true n_j x n_j part
      for (int i = 0; i < plan[bi].count; ++i) {
        const int n = dims[plan[bi].begin + i];
        max_n = std::max(max_n, n);
        sq += (size_t)n * n;
      }
      const size_t ld = (size_t)std::max(NOLSM_PAD, round_up(max_n, NOLSM_PAD));
      cache_sq[bi] = sq;
      cache_off[bi + 1] = cache_off[bi] + sq + (size_t)plan[bi].count * NOLSM_BS * ld;
    }
    size_t free_b = 0, total_b = 0;
    size_t cap = ctx->cfg.cache_bytes > 0 ? (size_t)ctx->cfg.cache_bytes : 0;
    if (cap == 0 && cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
      // everything that is free now, less the workspace bound (it may not be allocated yet) and 4 GiB
      const size_t reserve = ws + ((size_t)4 << 30);
      cap = free_b > reserve ? free_b - reserve : 0;
    }
    const size_t need = cache_off.back() * sizeof(float);
    if (need > 0 && need <= cap && cudaMalloc(&cache, need) != cudaSuccess) { cudaGetLastError(); cache = nullptr; }
  }

  cudaEvent_t tev[5];
  for (int i = 0; i < 5; ++i) cudaEventCreate(&tev[i]);
  // per batch: submatrices whose inverse / sign iteration did not converge (read after the step's synchronise)
  int32_t *h_flags = nullptr;
  if (cudaMallocHost(&h_flags, sizeof(int32_t) * 2 * std::max<size_t>(plan.size(), 1)) != cudaSuccess) {
    cudaGetLastError();
    for (int i = 0; i < 5; ++i) cudaEventDestroy(tev[i]);
    if (cache) cudaFree(cache);
    ctx->err = "allocation of the convergence flags failed";
    return NOLSM_ENOMEM;
  }
  auto cleanup = [&]() {
    for (int i = 0; i < 5; ++i) cudaEventDestroy(tev[i]);
    cudaStreamSynchronize(st);
    cudaFreeHost(h_flags);
    if (cache) cudaFree(cache);
  };
  int64_t inv_bad = 0, sign_bad = 0;

  double lo = mu_lo, hi = mu_hi, mu = 0.5 * (lo + hi), ne = 0.0;
  int step = 0;
  nolsm_status rc = NOLSM_OK;
  for (step = 0; step < max_steps; ++step) {
    mu = 0.5 * (lo + hi);
    if (cudaMemsetAsync(ctx->d_scalars, 0, 4 * sizeof(double), st) != cudaSuccess) { rc = NOLSM_ECUDA; break; }
    nolsm_sign_stats acc;
    memset(&acc, 0, sizeof(acc));
    acc.iter_min = 1 << 30;
    for (size_t bi = 0; bi < plan.size() && rc == NOLSM_OK; ++bi) {
      const Range &r = plan[bi];
      nolsm_batch *b = live[bi];
      const bool timed = stats != nullptr;
      if (timed) cudaEventRecord(tev[0], st);
      float *cache_b = cache ? cache + cache_off[bi] : nullptr;
      if (cache && step > 0) {
        // operands of this batch from the cache: B -> u3, own columns of S^-1 -> u2
        std::vector<int32_t> bd(dims.begin() + r.begin, dims.begin() + r.begin + r.count);
        rc = setup_batch(ctx, kOwnSlot, bd, r.begin, true, units, &b, st);
        if (rc != NOLSM_OK) break;
        const size_t slab_all = cache_sq[bi];
        ctx->launches += 2;
        // the padded part of u3 may hold anything: the sign stage only reads the true n x n part of B
        if (launch_pack_square(b, b->u[3], cache_b, false, st) != cudaSuccess) {
          ctx->err = "solve_mu: copy from the operator cache failed"; rc = NOLSM_ECUDA; break;
        }
        if (launch_own_columns(b, H->row_ptr, H->col_idx, b->u[2], cache_b + slab_all, false, st) != cudaSuccess) {
          ctx->err = "solve_mu: restoring the own columns of S^-1 failed"; rc = NOLSM_ECUDA; break;
        }
        b->engine_simt = false;
        b->prepared = true;
        b->prepared_precision = prec;
      } else if (!b || !resident) {
        // the FP32 copy of T_j(H) is only read by the energy products (nolsm_evaluate) and the SIMT debug path
        const bool need32 = ctx->eval_energy || use_simt(ctx) || !ctx->umma_ok;
        const bool fast32 = prec != NOLSM_FP16_FP32 && !ctx->eval_energy && ctx->inv_refine_default &&
                            (ctx->cfg.flags & NOLSM_FLAG_LOWDIN) == 0 &&
                            ctx->cfg.inv_tol <= 0.f && (ctx->cfg.flags & NOLSM_FLAG_NO_PREDICT) == 0;
        rc = build_submatrices_impl(ctx, H, S, r.begin, r.count, kOwnSlot + (resident ? (int)bi : 0), units, &b, st,
                                    need32, need32, fast32);
        if (rc != NOLSM_OK) break;
        live[bi] = resident ? b : nullptr;
      }
      if (timed) cudaEventRecord(tev[1], st);
      int64_t gemms = 0;
      nolsm_sign_stats bs;
      memset(&bs, 0, sizeof(bs));
      if (!b->prepared) {
        // a single N(mu) evaluation (the chemical potential is fixed): B itself is never needed
        const bool single = max_steps == 1 && !cache && !ctx->eval_energy;
        rc = prepare_batch(ctx, b, prec, st, stats ? &bs : nullptr, &gemms, !ctx->eval_energy, single ? &mu : nullptr);
        if (rc != NOLSM_OK) break;
        if (cache) {
          const size_t slab_all = cache_sq[bi];
          ctx->launches += 2;
          if (launch_pack_square(b, b->u[3], cache_b, true, st) != cudaSuccess) {
            ctx->err = "solve_mu: copy to the operator cache failed"; rc = NOLSM_ECUDA; break;
          }
          if (launch_own_columns(b, H->row_ptr, H->col_idx, b->u[2], cache_b + slab_all, true, st) != cudaSuccess) {
            ctx->err = "solve_mu: saving the own columns of S^-1 failed"; rc = NOLSM_ECUDA; break;
          }
        }
      }
      if (timed) cudaEventRecord(tev[2], st);
      // the last iteration is folded into the density columns unless W needs the iterate itself
      rc = sign_batch(ctx, b, mu, prec, tol, max_iter, fixed_iter, nullptr, st, timed, !ctx->eval_energy);
      if (rc != NOLSM_OK) break;
      if (timed) cudaEventRecord(tev[3], st);
      rc = nolsm_scatter_density(ctx, b, S, D, ctx->d_scalars, q_mol, ctx->d_scalars + 1, st);
      if (rc != NOLSM_OK) break;
      h_flags[2 * bi] = h_flags[2 * bi + 1] = 0;
      if (!b->engine_simt &&
          cudaMemcpyAsync(h_flags + 2 * bi, b->d_sched + 4, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess) {
        ctx->err = "solve_mu: copy of the convergence flags failed"; rc = NOLSM_ECUDA; break;
      }
      if (ctx->eval_energy) {   // nolsm_evaluate: E = Tr(D H0) and the own columns of W = D H0 D
        rc = nolsm_scatter_energy(ctx, b, H, D, ctx->eval_w, ctx->d_scalars + 2, st);
        if (rc != NOLSM_OK) break;
      }
      if (timed) {
        cudaEventRecord(tev[4], st);
        nolsm_sign_stats cs;
        memset(&cs, 0, sizeof(cs));
        rc = collect_stats(ctx, b, tol, fixed_iter, st, &cs);   // synchronises
        if (rc != NOLSM_OK) break;
        float ms[4];
        for (int i = 0; i < 4; ++i) cudaEventElapsedTime(&ms[i], tev[i], tev[i + 1]);
        stats->ms_gather += ms[0]; stats->ms_prepare += ms[1]; stats->ms_sign += ms[2]; stats->ms_density += ms[3];
        stats->ms_chain += chain_ms(ctx, b);
        stats->chain_launches += b->engine_simt ? 0 : 1;
        acc.n_sub += cs.n_sub;
        acc.iter_min = std::min(acc.iter_min, cs.iter_min);
        acc.iter_max = std::max(acc.iter_max, cs.iter_max);
        acc.iter_sum += cs.iter_sum;
        acc.n_unconverged += cs.n_unconverged;
        acc.worst_residual = std::max(acc.worst_residual, cs.worst_residual);
        acc.flops_sign += cs.flops_sign;
        acc.flops_sign_padded += cs.flops_sign_padded;
        acc.flops_prepare += bs.flops_prepare;
        acc.inv_iter_max = std::max(acc.inv_iter_max, bs.inv_iter_max);
        acc.gemms += gemms + b->sign_ops * cs.iter_sum - (b->x_pending ? b->count : 0);
      }
    }
    if (rc != NOLSM_OK) break;
    if (cudaMemcpyAsync(ctx->h_scalars, ctx->d_scalars, 4 * sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
      ctx->err = std::string("solve_mu: ") + cudaGetErrorString(cudaGetLastError());
      rc = NOLSM_ECUDA;
      break;
    }
    ne = ctx->h_scalars[0];
    sign_bad = 0;
    for (size_t bi = 0; bi < plan.size(); ++bi) {
      if (step == 0) inv_bad += h_flags[2 * bi];
      sign_bad += h_flags[2 * bi + 1];
    }
    if (stats) {
      stats->last = acc;
      stats->ne_diag = ctx->h_scalars[1];
      stats->flops_sign_total += acc.flops_sign;
      stats->flops_prepare_total += acc.flops_prepare;
      stats->mu_steps = step + 1;
    }
    if (!(ne == ne)) {
      if (inv_bad > 0) {
        ctx->err = std::to_string(inv_bad) + " submatrices: Eq. 15-17 did not converge (S_j not SPD?); N(mu) is NaN";
        rc = NOLSM_ENOTSPD;
      } else {
        ctx->err = "N(mu) is NaN";
        rc = NOLSM_ENOCONV;
      }
      break;
    }
    if (tol_ne_per_mol >= 0.0 && std::fabs(ne - n_electrons) <= tol_ne_per_mol * (double)n_mol) { step++; break; }
    if (step + 1 < max_steps) {
      if (ne > n_electrons) hi = mu; else lo = mu;
    }
  }
  cleanup();
  *mu_out = mu;
  *ne_out = ne;
  if (stats) {
    stats->n_batches = (int)plan.size();
    stats->resident = resident ? 1 : 0;
    stats->cached = cache ? 1 : 0;
    stats->mu_lo = lo;
    stats->mu_hi = hi;
    stats->last.n_unconverged = (int32_t)std::min<int64_t>(sign_bad, 0x7fffffff);
  }
  // The verdict does not depend on `stats` (the kernels count what did not converge):
  if (rc == NOLSM_OK && inv_bad > 0) {
    ctx->err = std::to_string(inv_bad) + " submatrices: Eq. 15-17 did not reach inv_tol within inv_max_iter (S_j not SPD?)";
    rc = NOLSM_ENOTSPD;
  } else if (rc == NOLSM_OK && sign_bad > 0 && fixed_iter <= 0) {
    ctx->err = std::to_string(sign_bad) + " submatrices: the sign iteration hit max_iter on the final mu";
    rc = NOLSM_ENOCONV;
  } else if (rc == NOLSM_OK && tol_ne_per_mol >= 0.0 && std::fabs(ne - n_electrons) > tol_ne_per_mol * (double)n_mol &&
             (lo == mu_lo || hi == mu_hi)) {
    // the bisection never moved one end of the bracket and did not meet the tolerance: N(mu) - N_e keeps one
    // sign over [mu_lo, mu_hi] as far as the midpoints can tell
    ctx->err = "no crossing of N(mu) = N_e found inside [mu_lo, mu_hi]";
    rc = NOLSM_EBRACKET;
  }
  return rc;
}

// One evaluation of the whole path at a given mu, with the electronic energy and (optionally) the
// energy-weighted density (Eq. 7, 8, 11, 13).
extern "C" nolsm_status nolsm_evaluate(nolsm_ctx *ctx, const nolsm_bsr *H, const nolsm_bsr *S, double mu,
                                       int32_t precision, nolsm_bsr *D, nolsm_bsr *W, double *ne_out, double *e_out,
                                       double *q_mol, nolsm_solve_stats *stats, void *stream) {
  if (!ctx || !ne_out || !e_out) return NOLSM_EINVAL;
  ctx->eval_energy = true;
  ctx->eval_w = W;
  double mu_found = 0.0;
  const double half = 1.0;   // bracket [mu - 1, mu + 1]: the first (and only) midpoint is mu itself
  nolsm_status rc = nolsm_solve_mu(ctx, H, S, 0.0, mu - half, mu + half, -1.0, 1, precision, D, &mu_found, ne_out,
                                   q_mol, stats, stream);
  ctx->eval_energy = false;
  ctx->eval_w = nullptr;
  *e_out = ctx->h_scalars[2];
  return rc;
}

// ------------------------------------------------------------------------------------------------
// Whole path with HOST buffers (end-to-end leg: transfers inside)
// ------------------------------------------------------------------------------------------------
extern "C" nolsm_status nolsm_solve_mu_host(nolsm_ctx *ctx, int32_t n_mol, const int32_t *row_ptr,
                                            const int32_t *col_idx, const float *h_val, const float *s_val,
                                            double n_electrons, double mu_lo, double mu_hi, double tol_ne_per_mol,
                                            int32_t max_steps, int32_t precision, float *d_val, double *mu_out,
                                            double *ne_out, nolsm_solve_stats *stats, int64_t *h2d_bytes,
                                            int64_t *d2h_bytes, void *stream) {
  if (!ctx) return NOLSM_EINVAL;
  if (n_mol <= 0 || !row_ptr || !col_idx || !h_val || !s_val || !d_val) {
    ctx->err = "nolsm_solve_mu_host: bad argument";
    return NOLSM_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t nnzb = row_ptr[n_mol];
  if (nnzb <= 0 || row_ptr[0] != 0) { ctx->err = "nolsm_solve_mu_host: bad row_ptr"; return NOLSM_EINVAL; }
  if ((size_t)n_mol > ctx->m_cap_mol) {
    cudaStreamSynchronize(st);
    cudaFree(ctx->m_row_ptr);
    ctx->m_row_ptr = nullptr;
    ctx->m_cap_mol = 0;
    if (cudaMalloc(&ctx->m_row_ptr, sizeof(int32_t) * ((size_t)n_mol + 1)) != cudaSuccess) {
      cudaGetLastError(); ctx->err = "cudaMalloc of the row_ptr mirror failed"; return NOLSM_ENOMEM;
    }
    ctx->m_cap_mol = (size_t)n_mol;
  }
  if ((size_t)nnzb > ctx->m_cap_nnzb) {
    cudaStreamSynchronize(st);
    cudaFree(ctx->m_col_idx); cudaFree(ctx->m_h); cudaFree(ctx->m_s); cudaFree(ctx->m_d);
    ctx->m_col_idx = nullptr; ctx->m_h = ctx->m_s = ctx->m_d = nullptr;
    ctx->m_cap_nnzb = 0;
    const size_t vb = sizeof(float) * 36 * (size_t)nnzb;
    if (cudaMalloc(&ctx->m_col_idx, sizeof(int32_t) * (size_t)nnzb) != cudaSuccess ||
        cudaMalloc(&ctx->m_h, vb) != cudaSuccess || cudaMalloc(&ctx->m_s, vb) != cudaSuccess ||
        cudaMalloc(&ctx->m_d, vb) != cudaSuccess) {
      cudaGetLastError(); ctx->err = "cudaMalloc of the block-store mirrors failed"; return NOLSM_ENOMEM;
    }
    ctx->m_cap_nnzb = (size_t)nnzb;
  }
  const size_t vb = sizeof(float) * 36 * (size_t)nnzb;
  NOLSM_CUDA(ctx, cudaMemcpyAsync(ctx->m_row_ptr, row_ptr, sizeof(int32_t) * ((size_t)n_mol + 1), cudaMemcpyHostToDevice, st));
  NOLSM_CUDA(ctx, cudaMemcpyAsync(ctx->m_col_idx, col_idx, sizeof(int32_t) * (size_t)nnzb, cudaMemcpyHostToDevice, st));
  NOLSM_CUDA(ctx, cudaMemcpyAsync(ctx->m_h, h_val, vb, cudaMemcpyHostToDevice, st));
  NOLSM_CUDA(ctx, cudaMemcpyAsync(ctx->m_s, s_val, vb, cudaMemcpyHostToDevice, st));
  nolsm_bsr H{n_mol, NOLSM_BS, ctx->m_row_ptr, ctx->m_col_idx, ctx->m_h};
  nolsm_bsr S{n_mol, NOLSM_BS, ctx->m_row_ptr, ctx->m_col_idx, ctx->m_s};
  nolsm_bsr D{n_mol, NOLSM_BS, ctx->m_row_ptr, ctx->m_col_idx, ctx->m_d};
  nolsm_status rc = nolsm_solve_mu(ctx, &H, &S, n_electrons, mu_lo, mu_hi, tol_ne_per_mol, max_steps, precision, &D,
                                   mu_out, ne_out, nullptr, stats, st);
  if (rc != NOLSM_OK && rc != NOLSM_ENOCONV) return rc;
  NOLSM_CUDA(ctx, cudaMemcpyAsync(d_val, ctx->m_d, vb, cudaMemcpyDeviceToHost, st));
  NOLSM_CUDA(ctx, cudaStreamSynchronize(st));
  if (h2d_bytes) *h2d_bytes = (int64_t)(2 * vb + sizeof(int32_t) * ((size_t)n_mol + 1 + (size_t)nnzb));
  if (d2h_bytes) *d2h_bytes = (int64_t)vb;
  return rc;
}

// ------------------------------------------------------------------------------------------------
// Dense microbench entry and the GEMM test entry
// ------------------------------------------------------------------------------------------------
extern "C" nolsm_status nolsm_sign_dense_batched(nolsm_ctx *ctx, const float *a, const float *scale, int32_t n,
                                                 int32_t batch, int32_t precision, float tol, int32_t max_iter,
                                                 int32_t fixed_iter, float *x_out, nolsm_sign_stats *stats,
                                                 void *stream) {
  if (!ctx || n <= 0 || batch < 0) return NOLSM_EINVAL;
  if (batch == 0) { if (stats) memset(stats, 0, sizeof(*stats)); return NOLSM_OK; }
  if (!a || !x_out) { ctx->err = "nolsm_sign_dense_batched: null matrix pointer"; return NOLSM_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const int prec = effective_precision(ctx, precision);
  resolve_sign_args(ctx, prec, &tol, &max_iter, &fixed_iter);
  if (stats) memset(stats, 0, sizeof(*stats));
  if (batch == 0) return NOLSM_OK;
  std::vector<int32_t> dims(batch, n);
  nolsm_batch *b = nullptr;
  CHECK(setup_batch(ctx, kOwnDense, dims, 0, false, units_dense(prec), &b, st));
  b->prepared = true;
  b->prepared_precision = prec;
  b->engine_simt = use_simt(ctx);
  LAUNCH(ctx, launch_pack(a, n, batch, b->ld, bmat_ptr(b), 0, st));
  CHECK(sign_batch(ctx, b, 0.0, prec, tol, max_iter, fixed_iter, scale, st, stats != nullptr));
  CHECK(join_x(ctx, b, st));
  LAUNCH(ctx, launch_unpack(x_ptr(b), b->ld, (int64_t)b->ld * b->ld, nullptr, nullptr, n, batch, x_out, st));
  if (stats) {
    CHECK(collect_stats(ctx, b, tol, fixed_iter, st, stats));
    stats->gemms = b->sign_ops * stats->iter_sum;
    stats->ms_chain = chain_ms(ctx, b);
    stats->chain_mcycles = chain_mcycles(ctx, b, st);
  }
  return NOLSM_OK;
}

extern "C" nolsm_status nolsm_batch_read(nolsm_ctx *ctx, const nolsm_batch *b, int32_t local, int32_t which,
                                         float *dst, int64_t dst_elems, int32_t *n_out, void *stream) {
  if (!ctx || !b || !dst || local < 0 || local >= b->count) return NOLSM_EINVAL;
  if (which == NOLSM_MAT_X && b->prepared) CHECK(join_x(ctx, const_cast<nolsm_batch *>(b), (cudaStream_t)stream));
  if (which == NOLSM_MAT_SINV && b->prepared) CHECK(join_sinv(ctx, const_cast<nolsm_batch *>(b), (cudaStream_t)stream));
  const int n = b->n_host[local];
  if (n_out) *n_out = n;
  if (dst_elems < (int64_t)n * n) { ctx->err = "dst too small"; return NOLSM_ENOMEM; }
  const float *src = nullptr;
  switch (which) {
    case NOLSM_MAT_S: src = b->u[0]; break;
    case NOLSM_MAT_H: src = b->u[1]; break;
    case NOLSM_MAT_SINV: src = b->prepared ? sinv_ptr(b) : nullptr; break;
    case NOLSM_MAT_B: src = b->prepared ? bmat_ptr(b) : nullptr; break;
    case NOLSM_MAT_X: src = b->prepared ? x_ptr(b) : nullptr; break;
    default: break;
  }
  if (!src) { ctx->err = "matrix not available in this batch state"; return NOLSM_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t slab = (int64_t)b->ld * b->ld;
  LAUNCH(ctx, launch_unpack(src + (int64_t)local * slab, b->ld, slab, nullptr, nullptr, n, 1, dst, st));
  NOLSM_CUDA(ctx, cudaStreamSynchronize(st));
  return NOLSM_OK;
}

extern "C" nolsm_status nolsm_gemm_batched(nolsm_ctx *ctx, int32_t kind, int32_t ident, float alpha, float beta,
                                           const float *a, const float *bm, const float *cin, float *c,
                                           float *resid2, int32_t n, int32_t batch, void *stream) {
  if (!ctx || !a || !bm || !c || n <= 0 || batch <= 0 || kind < 0 || kind > 3) return NOLSM_EINVAL;
  if (!ident && beta != 0.f && !cin) return NOLSM_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  std::vector<int32_t> dims(batch, n);
  nolsm_batch *b = nullptr;
  CHECK(setup_batch(ctx, kOwnDense, dims, 0, false, 7, &b, st));
  // unit padding in A and B keeps the padded rows/columns decoupled, like the iterates of the path
  LAUNCH(ctx, launch_pack(a, n, batch, b->ld, b->u[0], 1, st));
  LAUNCH(ctx, launch_pack(bm, n, batch, b->ld, b->u[1], 1, st));
  if (!ident && beta != 0.f) LAUNCH(ctx, launch_pack(cin, n, batch, b->ld, b->u[2], 0, st));
  const int mode = ident ? EPI_IDENT : EPI_AXPBY;
  float *resid_src = b->d_resid2;
  if (kind == 0) {
    Engine E{ctx, b, st};
    CHECK(E.zero_resid(0));
    CHECK(E.simt(mode, alpha, beta, nullptr, b->u[0], b->u[1], b->u[2], b->u[3], E.resid_slot(0), nullptr, 0));
  } else {
    LAUNCH(ctx, launch_scale_copy(b, b->u[0], nullptr, 0, nullptr, b->h[0], kind >= 2 ? b->h[1] : nullptr, st));
    LAUNCH(ctx, launch_scale_copy(b, b->u[1], nullptr, 0, nullptr, b->h[2], kind == 2 ? b->h[3] : nullptr, st));
    ChainProgram pg = one_shot(group_size(ctx, b, 16));
    pg.n_ops = 1;
    ChainOp &o = pg.ops[0] = make_op(mode, alpha, beta);
    set2(o.a, 0, 0); set2(o.b, 2, 2);
    if (kind >= 2) set2(o.a_lo, 1, 1);
    if (kind == 2) set2(o.b_lo, 3, 3);
    if (!ident && beta != 0.f) {
      if (kind == 3) {   // the add-in as a split FP16 pair through the staging buffers, like B1 = B0 + A0 R
        LAUNCH(ctx, launch_scale_copy(b, b->u[2], nullptr, 0, nullptr, b->h[4], b->h[5], st));
        set2(o.cin16, 4, 4); set2(o.cin16_lo, 5, 5);
      } else {
        o.cin32 = 2;
      }
    }
    o.cout32 = 3;
    o.resid = ident ? 1 : 0;
    CHECK(run_chain(ctx, b, pg, nullptr, true, st));
  }
  LAUNCH(ctx, launch_unpack(b->u[3], b->ld, (int64_t)b->ld * b->ld, nullptr, nullptr, n, batch, c, st));
  if (resid2 && ident)
    NOLSM_CUDA(ctx, cudaMemcpyAsync(resid2, resid_src, sizeof(float) * batch, cudaMemcpyDeviceToDevice, st));
  return NOLSM_OK;
}
