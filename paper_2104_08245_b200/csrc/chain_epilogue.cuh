// Epilogue and completion protocol of the matrix-iteration engine (chain_engine.cu), shared by its
// single-CTA and CTA-pair instantiations: one epilogue warp drains its 32 TMEM lanes (= 32 rows) of the
// tile in 32-column chunks, applies the fused epilogue of the op
//     EPI_IDENT :  E = I - A B,  ||E||_F^2 over the true n x n part (stop rule, reading 9)
//     EPI_AXPBY :  C = beta * C_in + alpha * A B   (master update, reading 12)
// and writes the FP32 result and/or the FP16 operand copies (hi [, lo * 2^11]).  The lanes of a warp hold
// consecutive rows of a column-major matrix, so every store instruction writes one contiguous 128-byte
// (FP32) or 64-byte (FP16) segment of a column.
//
// Completion protocol (rolling window, chain_engine.cu): after the stores of a tile the epilogue warps of
// the CTA meet at a named barrier and ONE elected thread makes them visible (__threadfence) and adds 1 to
// slot_done[s]; the arrival that completes the op evaluates the stop rule and publishes the slot's next
// state (same submatrix, next op -- or the next submatrix of the batch) with one 64-bit release store.
#pragma once
#include "common.cuh"

namespace chainep {

struct TileCmd {              // scheduler -> TMA producer(s), MMA issuer and epilogue warps (48 bytes)
  int32_t mat, m0, n0, nt;    // submatrix, first row / column of the tile, tile columns
  int32_t kblocks, ktail;     // K blocks of 64; K=16 steps in the last one (1..4)
  int32_t op, iter;           // op < 0: no more tiles
  int32_t slot, pad0, pad1, pad2;   // window slot the submatrix occupies
};

// TileCmd::iter carries the iteration in its low bits and, in bit 30, a flip of the operand-table parity
// (ChainProgram::parity_from_iters).
__device__ __forceinline__ int cmd_iter(const TileCmd &c) { return c.iter & 0x3fffffff; }
__device__ __forceinline__ int cmd_par(const TileCmd &c) { return (c.iter ^ (c.iter >> 30)) & 1; }

// Slot state word: round (24 bits) | ops of the submatrix already completed (8 bits) | submatrix (32 bits).
// A retired slot (no submatrix left to admit) holds kSlotDead: its round compares >= every round.
constexpr unsigned long long kSlotDead = 0xffffffffffffffffull;
__device__ __forceinline__ unsigned long long slot_pack(uint32_t round, uint32_t q, uint32_t mat) {
  return ((unsigned long long)round << 40) | ((unsigned long long)(q & 0xffu) << 32) | (unsigned long long)mat;
}
__device__ __forceinline__ uint32_t slot_round(unsigned long long s) { return (uint32_t)(s >> 40); }
__device__ __forceinline__ uint32_t slot_q(unsigned long long s) { return (uint32_t)(s >> 32) & 0xffu; }
__device__ __forceinline__ int32_t slot_mat(unsigned long long s) { return (int32_t)(uint32_t)s; }

struct ChainArgs {
  ChainProgram prog;
  const CUtensorMap *maps;    // [n_half] TMA maps of the FP16 operand buffers ({64,64} boxes, 128-byte swizzle)
  __half *hbuf[NOLSM_MAX_HALF];
  float *ubuf[NOLSM_MAX_UNIT];
  int32_t n_half, n_unit;
  int32_t count, ld;
  int64_t slab;
  int32_t bn, b_bytes, stages, stage_bytes;
  int32_t mt, ntl;            // uniform tile grid per submatrix: mt row tiles x ntl column tiles
  const int32_t *dims;
  const float *alpha_div;
  // rolling window of `window` submatrices
  int32_t window;
  unsigned long long *slot_state;     // [window]
  int32_t *slot_done;                 // [window] tiles of the slot's current op completed
  int32_t *sched;                     // [0] next submatrix to admit, [1] retired slots, [2] submatrices that hit max_iter,
                                      // [3] SM cycles / 1024 of the launch (max over CTAs; statistics)
  unsigned long long *tile_counter;   // next tile index to claim (dynamic, in-order scheduling)
  int32_t *state, *iters;
  float *resid2, *lastres;
  // op with colnorm, iteration k < colslots: colsum[k][count][ld] column sums of |E_k| (zero at launch; every thread
  // adds its rows' share and learns the running total), colmax[k][count] the largest running total seen = ||E_k||_1
  // once the product is complete (totals only grow)
  unsigned int *colsum;       // (fixed point, kColFix)
  unsigned int *colmax;
  int32_t colslots;
  // scaled Newton-Schulz start (nolsm_config.gap_hint): alpha_tab[m * kAlphaSteps + k] = alpha_k of submatrix m
  // for iteration k < kAlphaSteps (1 afterwards); null = the plain iteration
  const float *alpha_tab;
  // rescaled first sign iteration (ChainOp::colnorm == 2): alpha_rt[m], written when E_0 of submatrix m completes
  float *alpha_rt;
};
constexpr int kAlphaSteps = 8;
constexpr float kColFix = 1048576.f;   // column sums are accumulated as integers in units of 2^-20

__device__ __forceinline__ void ld_tmem32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, "
      "%22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]),
        "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]),
        "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]),
        "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr));
}
__device__ __forceinline__ void ld_tmem16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr));
}
__device__ __forceinline__ void ld_tmem_rows(uint32_t taddr, uint32_t (&v)[32]) { ld_tmem32(taddr, v); }
__device__ __forceinline__ void ld_tmem_rows(uint32_t taddr, uint32_t (&v)[16]) { ld_tmem16(taddr, v); }
__device__ __forceinline__ void ld_tmem_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void st_release_gpu_u64(unsigned long long *p, unsigned long long v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Called by ONE thread per CTA and tile after the CTA's epilogue warps have passed their barrier.
// kTileM / kColRound: tile rows and column rounding of the calling kernel (128 / 16 single-CTA,
// 256 / 32 pair); kArrivals: arrivals per tile (1, or 2 for a pair: one per CTA).
template <int kTileM, int kColRound, int kArrivals>
__device__ __forceinline__ void epi_complete(const ChainArgs &args, const TileCmd &c) {
  const ChainProgram &pg = args.prog;
  const ChainOp &o = pg.ops[c.op];
  const int n = args.dims[c.mat];
  const int ncol = (n + kColRound - 1) / kColRound * kColRound;
  const int tiles_m = ((n + kTileM - 1) / kTileM) * ((ncol + args.bn - 1) / args.bn);
  const int limit = pg.fixed_iter > 0 ? min(pg.fixed_iter, pg.max_iter) : pg.max_iter;
  __threadfence();      // the CTA's stores (ordered before us by the barrier) become visible GPU-wide
  const int32_t old = atomicAdd(&args.slot_done[c.slot], 1);
  if (old + 1 != tiles_m * kArrivals) return;
  __threadfence();
  const int k = cmd_iter(c);
  if (o.resid) {
    const float r2 = *reinterpret_cast<volatile float *>(
        &args.resid2[(size_t)(k % NOLSM_MAX_RESID_SLOTS) * args.count + c.mat]);
    const float res = (r2 == r2) ? sqrtf(fmaxf(r2, 0.f) / (float)n) : r2;   // fmaxf would swallow a NaN
    args.lastres[c.mat] = res;
    // ||E_k||_1 (E_k is symmetric: >= ||E_k||_2) as the epilogues left it: the largest running total of a column sum
    float pred = -1.f;
    if (o.colnorm == 1 && args.colsum != nullptr && k < args.colslots) {
      const float b1 = (float)*reinterpret_cast<volatile unsigned int *>(&args.colmax[(size_t)k * args.count + c.mat]) *
                       (1.f / kColFix);
      pred = b1 * b1 * (0.75f + 0.25f * b1);   // >= ||E_{k+1}||_2 (ChainProgram::tol_pred)
    }
    if (o.colnorm == 2 && k == 0 && args.colsum != nullptr && args.alpha_rt != nullptr) {
      // Rescaled first sign iteration (reading 5): rho(X0)^2 = rho(X0^2) <= ||X0^2||_1, known now.  X0 was
      // scaled so that the O(n^2) norm bound on rho maps to 1.5, which on these matrices is 1.8 x too careful; the
      // tighter bound is mapped to rescale_target (1.7 < sqrt 3, the edge of the convergence interval of Eq. 9) by
      // applying the step to a X0.  An eigenvalue that really sits at 1.7 lands at 0.09 and costs iterations, never the
      // limit; on these matrices the bound is 1.34 x off and the largest one lands at 0.88.  The 0.2 % cover the
      // operands' FP16 rounding (the product is of the hi parts) and the flooring of the fixed-point sums.
      const float b2 = 1.002f * (float)*reinterpret_cast<volatile unsigned int *>(&args.colmax[c.mat]) * (1.f / kColFix);
      float a = 1.f;
      // (not below one tile: nothing to save there, and with a handful of eigenvalues the stop residual has no
      // averaging -- an iterate taken right under the tolerance is then visibly less converged)
      if (b2 == b2 && b2 > 0.f && n >= NOLSM_TILE_M) a = pg.rescale_target * rsqrtf(fminf(b2, 2.25f));   // rho <= 1.5 holds in any case
      // a <= target: the update a (3/2 - 1/2 a^2) X0 + 1/2 a^3 X0 E_0 multiplies the FP16 rounding of E_0 by a^3, and
      // with a much larger a (a norm bound that was far off) it cancels catastrophically
      args.alpha_rt[c.mat] = fminf(fmaxf(a, 1.f), pg.rescale_target);
    }
    const bool conv = res < pg.tol;   // false for a NaN residual
    bool stop = pg.fixed_iter > 0 ? (k + 1 >= pg.fixed_iter) : (conv || !(res == res));
    // a scaled step (alpha_k > 1) measures ||I - alpha^2 X^2||, not the residual of the stop rule
    if (args.alpha_tab != nullptr && k < kAlphaSteps && pg.fixed_iter <= 0 && res == res &&
        args.alpha_tab[c.mat * kAlphaSteps + k] > 1.f)
      stop = false;
    if (k + 1 >= pg.max_iter) stop = true;
    // ended by the cap or by a NaN, not by a passing residual: the submatrix counts as not converged
    if (stop && pg.fixed_iter <= 0 && !conv) atomicAdd(&args.sched[2], 1);
    args.iters[c.mat] = (stop && pg.stop_early) ? k : k + 1;   // iterations carried out in full
    // state word: iteration that ends the chain | last op of that iteration << 24 (stop_early programs)
    if (stop) {
      *reinterpret_cast<volatile int32_t *>(&args.state[c.mat]) = k;
    } else if (pg.tol_pred > 0.f && pg.stop_early && pg.fixed_iter <= 0 && res == res && pred >= 0.f &&
               pred <= pg.tol_pred) {
      // a-priori stop: the bound on the NEXT residual passes, so iteration k only forms Z_{k+1} (op 1)
      args.lastres[c.mat] = pred;
      *reinterpret_cast<volatile int32_t *>(&args.state[c.mat]) = k | (1 << 24);
    }
  }
  const int32_t stv = *reinterpret_cast<volatile int32_t *>(&args.state[c.mat]);
  const bool stopping = (stv & 0xffffff) == k;
  // stop_early: the residual product is op 0 and the remaining products of a passing iteration are not run
  // (a-priori stop: those after op 1)
  const int last_op = !stopping ? pg.n_ops - 1 : (pg.stop_early ? ((stv >> 24) & 0x7f) : pg.n_ops - 1 - pg.skip_tail);
  const unsigned long long cur = *reinterpret_cast<volatile unsigned long long *>(&args.slot_state[c.slot]);
  const uint32_t round = slot_round(cur);
  args.slot_done[c.slot] = 0;
  unsigned long long next;
  if ((stopping && c.op == last_op) || (c.op == pg.n_ops - 1 && k + 1 >= limit)) {
    // this submatrix is finished: the slot admits the next one of the batch, or retires
    const int32_t m2 = atomicAdd(&args.sched[0], 1);
    if (m2 < args.count) {
      next = slot_pack(round + 1, 0, (uint32_t)m2);
    } else {
      next = kSlotDead;
      atomicAdd(&args.sched[1], 1);
    }
  } else {
    next = slot_pack(round + 1, slot_q(cur) + 1, (uint32_t)c.mat);
  }
  __threadfence();
  st_release_gpu_u64(&args.slot_state[c.slot], next);
}

// ------------------------------------------------------------------------------------------------
// Staged epilogue.  The engine computes the transposed product (chain_engine.cu), so TMEM lane = COLUMN of the
// result and TMEM column = ROW: after tcgen05.ld a thread holds 32 consecutive elements of one column, i.e. 64
// contiguous bytes of the column-major FP16 buffers.  Every FP16 stream of the epilogue -- the FP16 add-in
// (master hi [+ lo]) and the FP16 outputs (operand copies hi [+ lo]) -- moves between global memory and a
// shared-memory staging buffer by TMA (boxes of 64 rows x 128 columns, 128-byte swizzle, issued by ONE agent
// thread), and the compute warps touch the staging planes with 16-byte accesses only.  (Per-lane 2-byte global
// accesses cost the SM's L2 port as much per request as 4-byte ones, and 2-byte shared-memory accesses made the
// epilogue LSU-issue-bound: measured.)  FP32 streams (one-shot products of the prepare stage) stay on the
// direct path: 128 contiguous bytes per thread, 16-byte accesses.
//
// The eight compute warps (TMEM lane quadrant q = warp % 4 -> 32 columns of the tile, row half h = 32 rows)
// work through the tile in chunks of 64 rows; two staging buffers of two planes (hi, lo); plane = [128 columns][64 rows] FP16
// = 128 bytes per column, 16-byte pieces XOR-swizzled with (column % 8) like the TMA box.
// Protocol per chunk and buffer:
//   agent:    buffer free (its last store has been read) -> TMA loads of the add-in, or a plain arrive -> in_full
//   compute:  tcgen05.ld; wait in_full; add-in from smem; results into the SAME smem positions; fence; -> out_ready
//   agent:    wait out_ready; TMA stores; commit
// After the last chunk of a tile the agent waits for its stores to complete, waits for the compute warps
// (tile_done: their direct stores and residual atomics are issued) and publishes the tile (epi_complete).
// ------------------------------------------------------------------------------------------------
constexpr int kChunkRows = 64;
constexpr int kPlaneBytes = 128 * kChunkRows * 2;  // one FP16 plane of a chunk
constexpr int kStageBufBytes = 2 * kPlaneBytes;    // hi + lo
constexpr int kStagingBytes = 2 * kStageBufBytes;  // two buffers
constexpr int kComputeWarps = 8;                   // 4 lane quadrants x 2 row halves of a chunk (16 warps with 16 rows
                                                   // each measured 9 % slower: more barrier traffic, narrower accesses)
constexpr int kWarpRows = kChunkRows * 4 / kComputeWarps;   // rows of a chunk one warp drains: 32

struct EpiBars {
  uint64_t in_full[2], out_ready[2];
  uint64_t tile_done[2];   // by tile parity: the agent opens at most one tile ahead of the one it publishes, so the
                           // compute warps can never be two phases ahead of it on one barrier
};

__device__ __forceinline__ uint32_t s32(const void *p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void ebar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "EWAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra EWAIT_DONE;\n\t"
      "bra EWAIT_LOOP;\n\t"
      "EWAIT_DONE:\n\t"
      "}\n" ::"r"(s32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void ebar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(s32(bar)) : "memory");
}
__device__ __forceinline__ void ebar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_box(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(s32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(s32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ void tma_store_box(const void *src, const CUtensorMap *map, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(
                   reinterpret_cast<uint64_t>(map)),
               "r"(s32(src)), "r"(c0), "r"(c1), "r"(c2)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// What a tile's op moves through the staging buffers (the same for the agent and the compute warps)
struct EpiIO {
  int in_hi, in_lo, out_hi, out_lo;   // FP16 buffer indices, -1: none
  int out32;                          // FP32 unit written THROUGH the staging buffer (an op without FP16 outputs:
                                      // plane 0 / plane 1 hold rows 0..31 / 32..63 of the chunk as FP32), -1: none
  int nchunks;                        // chunks of 64 rows
};
__device__ __forceinline__ EpiIO epi_io(const ChainArgs &args, const TileCmd &c) {
  const ChainOp &o = args.prog.ops[c.op];
  const int par = cmd_par(c);
  EpiIO io;
  const bool ident = o.mode == EPI_IDENT;
  const bool cin = !ident && o.beta != 0.f && o.cin16[par] >= 0;
  io.in_hi = cin ? o.cin16[par] : -1;
  io.in_lo = cin ? o.cin16_lo[par] : -1;
  io.out_hi = o.out16[par];
  io.out_lo = o.out16_lo[par];
  io.out32 = (o.cout32 >= 0 && io.out_hi < 0) ? o.cout32 : -1;
  io.nchunks = (c.nt + kChunkRows - 1) / kChunkRows;
  return io;
}

// ---- the agent: one thread ----
// emaps: the {64 rows x 128 columns} box maps of the FP16 buffers; stage: the two staging buffers; col0: first
// column of this CTA's part of the tile; uses[b]: completed uses of buffer b (barrier phases).
__device__ __forceinline__ void epi_agent_avail(const TileCmd &c, const EpiIO &io, const CUtensorMap *emaps,
                                                uint8_t *stage, EpiBars &bars, int col0, int j) {
  const int b = j & 1;
  uint8_t *buf = stage + b * kStageBufBytes;
  const int row = c.n0 + kChunkRows * j;
  if (io.in_hi >= 0) {
    ebar_expect_tx(&bars.in_full[b], (uint32_t)kPlaneBytes * (io.in_lo >= 0 ? 2u : 1u));
    tma_load_box(buf, &emaps[io.in_hi], &bars.in_full[b], row, col0, c.mat);
    if (io.in_lo >= 0) tma_load_box(buf + kPlaneBytes, &emaps[io.in_lo], &bars.in_full[b], row, col0, c.mat);
  } else {
    ebar_arrive(&bars.in_full[b]);
  }
}
// Opens a tile: both staging buffers are free; the first two chunks become available to the compute warps.
__device__ __forceinline__ void epi_agent_open(const ChainArgs &args, const TileCmd &c, const CUtensorMap *emaps,
                                               uint8_t *stage, EpiBars &bars, int col0) {
  const EpiIO io = epi_io(args, c);
  if (io.nchunks > 0) epi_agent_avail(c, io, emaps, stage, bars, col0, 0);
  if (io.nchunks > 1) epi_agent_avail(c, io, emaps, stage, bars, col0, 1);
}
// Stores every chunk of an opened tile; on return all stores have READ their staging buffers (both are free),
// but may not be complete yet (bulk_wait0).
__device__ __forceinline__ void epi_agent_run(const ChainArgs &args, const TileCmd &c, const CUtensorMap *emaps,
                                              uint8_t *stage, EpiBars &bars, int col0, uint32_t (&uses)[2]) {
  const EpiIO io = epi_io(args, c);
  const int nch = io.nchunks;
  for (int j = 0; j < nch; ++j) {
    const int b = j & 1;
    ebar_wait(&bars.out_ready[b], uses[b] & 1u);
    ++uses[b];
    const uint8_t *buf = stage + b * kStageBufBytes;
    const int row = c.n0 + kChunkRows * j;
    if (io.out_hi >= 0) tma_store_box(buf, &emaps[io.out_hi], row, col0, c.mat);
    if (io.out_lo >= 0) tma_store_box(buf + kPlaneBytes, &emaps[io.out_lo], row, col0, c.mat);
    if (io.out32 >= 0) {   // FP32 maps follow the FP16 ones: {32 rows x 128 columns} boxes
      tma_store_box(buf, &emaps[args.n_half + io.out32], row, col0, c.mat);
      tma_store_box(buf + kPlaneBytes, &emaps[args.n_half + io.out32], row + 32, col0, c.mat);
    }
    bulk_commit();
    if (j + 2 < nch) {
      bulk_wait_read0();     // the store just issued has read the buffer: it may take the next add-in
      epi_agent_avail(c, io, emaps, stage, bars, col0, j + 2);
    }
  }
  bulk_wait_read0();
}

// ---- compute warp: cached per-tile parameters ----
struct EpiTile {
  const ChainOp *o;
  int par, n, col, h;         // col: this thread's column of the result; h: row quarter of every chunk
  bool split, ident, cin_direct, colnorm;
  bool norm_product;          // colnorm sums |alpha * accumulator| (the product itself) instead of |result|
  float alpha, beta, diag;
  float abs_sum;              // colnorm: sum of |result| over this thread's rows of the tile (true n x n part)
  float *p32;                 // FP32 output, element (first row of this warp's quarter, col) or null
  const float *cinp;          // FP32 master input (direct path), same position, or null
  EpiIO io;
  float cpre[kWarpRows];      // direct path only: add-in of the next chunk
};

__device__ __forceinline__ void epi_prefetch32(EpiTile &t) {
  const float4 *pc = reinterpret_cast<const float4 *>(t.cinp);
#pragma unroll
  for (int j = 0; j < kWarpRows / 4; ++j) {
    const float4 x = __ldcg(pc + j);
    t.cpre[4 * j] = x.x; t.cpre[4 * j + 1] = x.y; t.cpre[4 * j + 2] = x.z; t.cpre[4 * j + 3] = x.w;
  }
}

// Before waiting for the accumulator.  col: this thread's column of the result; h: row quarter of the chunks.
// kFeat: the epilogue / operand features the kernel instantiation supports (chain_engine.cu: program_features picks the
// smallest instantiation that covers a program).  The compute warps' code decides the kernel's register budget, and a
// feature that is compiled in costs the sign iteration 0.5-3 % even though it never runs there; with a feature bit
// clear its flag below is a compile-time constant and the code drops out of the kernel.
constexpr int kFeatSplitAny = 1;    // products may have split operands (full or half split), decided per op
constexpr int kFeatSplitAll = 2;    // every product is a full-split product
constexpr int kFeatColNorm = 4;     // column norms of the residual product (a-priori stop of Eq. 15-17)
constexpr int kFeatShift = 8;       // diagonal shift, per-matrix division of beta and the shift (X0 from B1's epilogue)
constexpr int kFeatFp32 = 16;       // FP32 inputs / outputs (direct or through the staging buffers)
constexpr int kFeatAlphaTab = 32;   // per-iteration scaling table (nolsm_config.gap_hint)
constexpr int kFeatRescale = 64;    // first sign iteration rescaled from ||X0^2||_1 (ChainOp::colnorm == 2)
constexpr int kFeatFull = 127 & ~kFeatSplitAll;
template <int kFeat>
__device__ __forceinline__ void epi_begin(const ChainArgs &args, const TileCmd &c, int col, int h, EpiTile &t) {
  const ChainOp &o = args.prog.ops[c.op];
  t.o = &o;
  t.par = cmd_par(c);
  t.n = args.dims[c.mat];
  t.col = col;
  t.h = h;
  t.io = epi_io(args, c);
  t.ident = o.mode == EPI_IDENT;
  t.abs_sum = 0.f;
  t.alpha = o.use_div ? o.alpha / args.alpha_div[c.mat] : o.alpha;
  float rescale_beta = 1.f;
  if constexpr ((kFeat & kFeatSplitAll) != 0) t.split = true;
  else if constexpr ((kFeat & kFeatSplitAny) != 0) t.split = o.a_lo[t.par] >= 0;
  else t.split = false;
  t.norm_product = false;
  if constexpr ((kFeat & kFeatColNorm) != 0) t.colnorm = t.ident && o.colnorm == 1;
  else t.colnorm = false;
  if constexpr ((kFeat & kFeatRescale) != 0) {
    if (o.colnorm == 2 && cmd_iter(c) == 0) {
      if (t.ident) {
        t.colnorm = t.norm_product = true;         // E_0 = I - X0^2: column sums of |X0^2|
      } else {
        // X_1 = a X0 (I + 1/2 (I - a^2 X0^2)) = a (3/2 - 1/2 a^2) X0 + 1/2 a^3 X0 E_0, a from E_0's completion
        const float a = *reinterpret_cast<volatile float *>(&args.alpha_rt[c.mat]);
        t.alpha *= a * a * a;
        rescale_beta = a * (1.5f - 0.5f * a * a);
      }
    }
  }
  if constexpr ((kFeat & kFeatShift) != 0) {
    t.beta = o.use_div == 2 ? o.beta / args.alpha_div[c.mat] : o.beta;
    t.diag = o.use_div == 2 ? o.diag / args.alpha_div[c.mat] : o.diag;
  } else {
    t.beta = o.beta;
    t.diag = 0.f;
  }
  t.beta *= rescale_beta;
  if constexpr ((kFeat & kFeatAlphaTab) != 0) {
    if (args.alpha_tab != nullptr && cmd_iter(c) < kAlphaSteps) {
      // X_{k+1} = 1/2 a X (3I - a^2 X^2):  E = I - a^2 X X,  X' = a X + (1/2 a) X E
      const float a = args.alpha_tab[c.mat * kAlphaSteps + cmd_iter(c)];
      if (t.ident) t.alpha *= a * a; else { t.alpha *= a; t.beta *= a; }
    }
  }
  if constexpr ((kFeat & kFeatFp32) != 0) {
    t.cin_direct = !t.ident && o.cin32 >= 0 && o.beta != 0.f && t.io.in_hi < 0;
    const int64_t off = (int64_t)c.mat * args.slab + (int64_t)col * args.ld + c.n0 + kWarpRows * h;
    t.p32 = (o.cout32 >= 0 && t.io.out32 < 0) ? args.ubuf[o.cout32] + off : nullptr;
    t.cinp = t.cin_direct ? args.ubuf[o.cin32] + off : nullptr;
    if (t.cin_direct && kWarpRows * h < c.nt) epi_prefetch32(t);
  } else {
    t.io.out32 = -1;
    t.cin_direct = false;
    t.p32 = nullptr;
    t.cinp = nullptr;
  }
}

// ------------------------------------------------------------------------------------------------
// Straight-line versions of epi_chunks for the two products that carry > 90 % of the work, the sign iteration in
// FP16/FP32 mode (and the residual product of Eq. 15-17):
//   kIdent = true :  E = I - alpha A B, FP16 result (hi only), ||E||_F^2            (EPI_IDENT, plain operands)
//   kIdent = false:  X' = beta (hi + lo/2048) + alpha A B, result as hi + lo        (EPI_AXPBY, split master)
// Same protocol and staging layout as epi_chunks; no per-element predicates or branches: ragged chunks, rows beyond
// the true dimension and chunks that hold diagonal elements are detected per warp and take the general code.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool epi_fast_kind(const EpiTile &t, bool &ident) {
  ident = t.ident;
  if (t.split || t.p32 != nullptr || t.cin_direct || kWarpRows != 32) return false;
  if (t.ident) return t.io.out_hi >= 0 && t.io.out_lo < 0;
  return t.io.in_hi >= 0 && t.io.out_hi >= 0 && t.io.out_lo >= 0;   // a diagonal shift: chunks off the diagonal only
}

template <bool kIdent, bool kInLo = true, bool kNorm = false>
__device__ __forceinline__ void epi_chunk_fast(const TileCmd &c, const EpiTile &t, uint32_t (&v)[32], uint8_t *hi_col,
                                               uint8_t *lo_col, int sw, float beta_lo, float &ss, float *sa = nullptr) {
  if constexpr (kIdent) {
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      uint32_t hw[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int jj = 8 * p + 2 * e;
        const float ea = -t.alpha * __uint_as_float(v[jj]), eb = -t.alpha * __uint_as_float(v[jj + 1]);
        ss = fmaf(ea, ea, ss);
        ss = fmaf(eb, eb, ss);
        if constexpr (kNorm) *sa += fabsf(ea) + fabsf(eb);
        const __half2 h2 = __floats2half2_rn(ea, eb);
        hw[e] = *reinterpret_cast<const uint32_t *>(&h2);
      }
      *reinterpret_cast<uint4 *>(hi_col + (((4 * t.h + p) ^ sw) * 16)) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
    }
  } else {
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      const int pc = ((4 * t.h + p) ^ sw) * 16;
      const uint4 hq = *reinterpret_cast<const uint4 *>(hi_col + pc);
      uint4 lq = make_uint4(0u, 0u, 0u, 0u);
      if constexpr (kInLo) lq = *reinterpret_cast<const uint4 *>(lo_col + pc);
      const uint32_t hin[4] = {hq.x, hq.y, hq.z, hq.w}, lin[4] = {lq.x, lq.y, lq.z, lq.w};
      uint32_t hw[4], lw[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int jj = 8 * p + 2 * e;
        const float2 hf = __half22float2(*reinterpret_cast<const __half2 *>(&hin[e]));
        const float2 lf = __half22float2(*reinterpret_cast<const __half2 *>(&lin[e]));
        const float xa = fmaf(t.alpha, __uint_as_float(v[jj]), kInLo ? fmaf(beta_lo, lf.x, t.beta * hf.x) : t.beta * hf.x);
        const float xb = fmaf(t.alpha, __uint_as_float(v[jj + 1]), kInLo ? fmaf(beta_lo, lf.y, t.beta * hf.y) : t.beta * hf.y);
        const __half2 h2 = __floats2half2_rn(xa, xb);
        const float2 hb = __half22float2(h2);
        const __half2 l2 = __floats2half2_rn((xa - hb.x) * 2048.f, (xb - hb.y) * 2048.f);
        hw[e] = *reinterpret_cast<const uint32_t *>(&h2);
        lw[e] = *reinterpret_cast<const uint32_t *>(&l2);
      }
      *reinterpret_cast<uint4 *>(hi_col + pc) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
      *reinterpret_cast<uint4 *>(lo_col + pc) = make_uint4(lw[0], lw[1], lw[2], lw[3]);
    }
  }
}


// Drains this warp's 16 rows of every chunk of the accumulator at TMEM address t_main (lane quadrant and
// accumulator stage already applied).  stage: the staging buffers; cl: this thread's column inside the CTA's part
// of the tile (0..127); uses[b]: completed uses of buffer b.  Tile heights are multiples of 16, so a warp's part
// of a chunk is complete, half (16 rows) or empty.  Returns the warp's partial residual sum (lane-local; reduce before use).
// release(): called once, as soon as this warp's last accumulator rows of the tile are in registers (the MMA issuer
// may then reuse the accumulator stage while the last chunk is still being processed).
template <typename Release>
__device__ __forceinline__ float epi_chunks(const ChainArgs &args, const TileCmd &c, EpiTile &t, uint32_t t_main,
                                            int lane, int cl, uint8_t *stage, EpiBars &bars, uint32_t (&uses)[2],
                                            Release release) {
  constexpr int R = kWarpRows;
  float ss = 0.f;
  const int sw = cl & 7;                          // XOR swizzle of the 16-byte pieces of this column
  const int scol = cl * (2 * kChunkRows);         // byte offset of this column inside a staging plane
  const float beta_lo = t.beta * (1.f / 2048.f);
  bool fast_ident = false;
  const bool fast_kind = epi_fast_kind(t, fast_ident);
  uint32_t va[R], vb[R];
  // plain products: the accumulator rows of chunk i + 1 are fetched from TMEM while chunk i is processed
  if (!t.split && R * t.h < c.nt) ld_tmem_rows(t_main + R * t.h, va);
  auto chunk = [&](const int ci, uint32_t (&v)[R], uint32_t (&vnext)[R]) {
    const int b = ci & 1;
    const int c0 = ci * kChunkRows + R * t.h;     // first row (inside the tile) of this warp's part of the chunk
    const int cnt = max(0, min(R, c.nt - c0));    // valid rows: R, 16 or 0
    const bool live = cnt > 0;
    if (t.split) {
      if (live) {
        uint32_t w[R];
        ld_tmem_rows(t_main + c0, v);
        ld_tmem_rows(t_main + 128 + c0, w);
        ld_tmem_wait();
#pragma unroll
        for (int jj = 0; jj < R; ++jj)
          v[jj] = __float_as_uint(fmaf(__uint_as_float(w[jj]), 1.f / 2048.f, __uint_as_float(v[jj])));
      }
    } else {
      ld_tmem_wait();
      if (c0 + kChunkRows < c.nt) ld_tmem_rows(t_main + c0 + kChunkRows, vnext);
    }
    if (ci == t.io.nchunks - 1) release();
    // the staging buffer is free (its previous store has been read) and holds this chunk's add-in, if any
    ebar_wait(&bars.in_full[b], uses[b] & 1u);
    ++uses[b];
    uint8_t *hi_col = stage + b * kStageBufBytes + scol;
    uint8_t *lo_col = hi_col + kPlaneBytes;
    if constexpr (R == 32) {
      // straight-line code for the products of the sign iteration (epi_chunk_fast) when the warp's part of the
      // chunk is complete, inside the true dimension and (residual product) holds no diagonal element
      bool fast = fast_kind && cnt == R;
      if (fast && (fast_ident || t.diag != 0.f)) {
        const int dj = t.col - (c.n0 + c0);
        fast = (!fast_ident || c.n0 + c0 + R <= t.n) && !__any_sync(0xffffffffu, dj >= 0 && dj < R);
      }
      if (fast) {
        float s_local = 0.f, a_local = 0.f;
        if (fast_ident && t.colnorm) epi_chunk_fast<true, true, true>(c, t, v, hi_col, lo_col, sw, beta_lo, s_local, &a_local);
        else if (fast_ident) epi_chunk_fast<true>(c, t, v, hi_col, lo_col, sw, beta_lo, s_local);
        else if (t.io.in_lo >= 0) epi_chunk_fast<false, true>(c, t, v, hi_col, lo_col, sw, beta_lo, s_local);
        else epi_chunk_fast<false, false>(c, t, v, hi_col, lo_col, sw, beta_lo, s_local);
        if (t.col < t.n) { ss += s_local; t.abs_sum += a_local; }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) ebar_arrive(&bars.out_ready[b]);
        return;
      }
    }
    if (live) {
      if (t.io.in_hi >= 0) {
        const bool has_lo = t.io.in_lo >= 0;
#pragma unroll
        for (int p = 0; p < R / 8; ++p) {
          const int pc = (((R / 8) * t.h + p) ^ sw) * 16;
          const uint4 hq = *reinterpret_cast<const uint4 *>(hi_col + pc);
          uint4 lq = make_uint4(0u, 0u, 0u, 0u);
          if (has_lo) lq = *reinterpret_cast<const uint4 *>(lo_col + pc);
          const uint32_t hw[4] = {hq.x, hq.y, hq.z, hq.w}, lw[4] = {lq.x, lq.y, lq.z, lq.w};
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float2 hf = __half22float2(*reinterpret_cast<const __half2 *>(&hw[e]));
            const float2 lf = __half22float2(*reinterpret_cast<const __half2 *>(&lw[e]));
            const int jj = 8 * p + 2 * e;
            // beta (hi + lo / 2048) + alpha v
            v[jj] = __float_as_uint(fmaf(t.alpha, __uint_as_float(v[jj]), fmaf(beta_lo, lf.x, t.beta * hf.x)));
            v[jj + 1] = __float_as_uint(fmaf(t.alpha, __uint_as_float(v[jj + 1]), fmaf(beta_lo, lf.y, t.beta * hf.y)));
          }
        }
      } else if (t.cin_direct) {
#pragma unroll
        for (int jj = 0; jj < R; ++jj)
          v[jj] = __float_as_uint(fmaf(t.beta, t.cpre[jj], t.alpha * __uint_as_float(v[jj])));
        if (c0 + kChunkRows < c.nt) {
          t.cinp += kChunkRows;
          epi_prefetch32(t);
        }
      } else if (t.ident) {
        // valid rows of this chunk inside the true n x n part (residual of the stop rule)
        const int nvalid = (t.col < t.n) ? min(cnt, t.n - (c.n0 + c0)) : 0;
        const int dj = t.col - (c.n0 + c0);   // chunk row that holds the diagonal element of this column
#pragma unroll
        for (int jj = 0; jj < R; ++jj) {
          const float e = fmaf(-t.alpha, __uint_as_float(v[jj]), (jj == dj) ? 1.f : 0.f);
          if (jj < nvalid) {
            ss = fmaf(e, e, ss);
            if (t.colnorm) t.abs_sum += t.norm_product ? fabsf(t.alpha * __uint_as_float(v[jj])) : fabsf(e);
          }
          v[jj] = __float_as_uint(e);
        }
      } else {
#pragma unroll
        for (int jj = 0; jj < R; ++jj) v[jj] = __float_as_uint(t.alpha * __uint_as_float(v[jj]));
      }
      if (t.diag != 0.f && !t.ident) {   // + diag * I: the chunk row that holds the diagonal element of this column
        const int dj = t.col - (c.n0 + c0);
#pragma unroll
        for (int jj = 0; jj < R; ++jj)
          if (jj == dj) v[jj] = __float_as_uint(__uint_as_float(v[jj]) + t.diag);
      }
      if (t.p32) {   // FP32 result (direct): 64 contiguous bytes of this thread's column
        float4 *qp = reinterpret_cast<float4 *>(t.p32);
#pragma unroll
        for (int j4 = 0; j4 < R / 4; ++j4)
          if (4 * j4 < cnt)
            qp[j4] = make_float4(__uint_as_float(v[4 * j4]), __uint_as_float(v[4 * j4 + 1]),
                               __uint_as_float(v[4 * j4 + 2]), __uint_as_float(v[4 * j4 + 3]));
        t.p32 += kChunkRows;
      }
    }
    // an FP32 result over an FP16 add-in: the result of row half h fills all of plane h, which holds add-in pieces
    // of the other half's warps, so every compute warp has to have read its add-in first (all of them pass here:
    // the chunk loop and the branches above are uniform over the compute warps)
    if (t.io.out32 >= 0 && t.io.in_hi >= 0) asm volatile("bar.sync 1, %0;" ::"n"(kComputeWarps * 32) : "memory");
    if (t.io.out32 >= 0) {    // FP32 result into the plane of this warp's row half; rows beyond the tile as zero
      if (cnt < R) {
#pragma unroll
        for (int jj = 0; jj < R; ++jj)
          if (jj >= cnt) v[jj] = 0u;
      }
      uint8_t *pl = hi_col + t.h * kPlaneBytes;
#pragma unroll
      for (int p = 0; p < R / 4; ++p)
        *reinterpret_cast<uint4 *>(pl + ((p ^ sw) * 16)) = make_uint4(v[4 * p], v[4 * p + 1], v[4 * p + 2], v[4 * p + 3]);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (t.io.out_hi >= 0) {   // FP16 copies into the staging planes; rows beyond the tile are written as zero
      const bool has_lo = t.io.out_lo >= 0;
      if (cnt < R) {          // ragged last chunk (warp-uniform, rare)
#pragma unroll
        for (int jj = 0; jj < R; ++jj)
          if (jj >= cnt) v[jj] = 0u;
      }
#pragma unroll
      for (int p = 0; p < R / 8; ++p) {
        uint32_t hw[4], lw[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int jj = 8 * p + 2 * e;
          const float va_ = __uint_as_float(v[jj]), vb_ = __uint_as_float(v[jj + 1]);
          const __half2 h2 = __floats2half2_rn(va_, vb_);
          hw[e] = *reinterpret_cast<const uint32_t *>(&h2);
          const float2 hf = __half22float2(h2);
          const __half2 l2 = __floats2half2_rn((va_ - hf.x) * 2048.f, (vb_ - hf.y) * 2048.f);
          lw[e] = *reinterpret_cast<const uint32_t *>(&l2);
        }
        const int pc = (((R / 8) * t.h + p) ^ sw) * 16;
        *reinterpret_cast<uint4 *>(hi_col + pc) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
        if (has_lo) *reinterpret_cast<uint4 *>(lo_col + pc) = make_uint4(lw[0], lw[1], lw[2], lw[3]);
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy smem writes -> TMA store
    }
    __syncwarp();
    if (lane == 0) ebar_arrive(&bars.out_ready[b]);
  };
  for (int ci = 0; ci < t.io.nchunks; ci += 2) {
    chunk(ci, va, vb);
    if (ci + 1 < t.io.nchunks) chunk(ci + 1, vb, va);
  }
  return ss;
}

}  // namespace chainep
