// The batched matrix-iteration engine: ONE persistent, cooperative kernel runs a whole chain of
// dependent n x n x n products (every iteration of Eq. 9-10, or of Eq. 15-17
// PAPER.md:203-215) for every submatrix of a batch on the 5th-generation tensor cores
// (tcgen05 + TMEM + TMA), sm_100a only.
//
// Why one kernel: the two products of a sign iteration are strictly dependent and one product of an
// n ~ 860 submatrix is < 1 us of the whole GPU, so kernel boundaries would cost more than the work, and
// a batch-wide launch per product streams every iterate through HBM (18 n^2 bytes per 4 n^3 FLOP,
// DESIGN.md "Roofline").  The submatrices are walked in GROUPS, each iterated to convergence before the
// next is touched (the B200 analogue of the paper's "caching strategy for the matrices during the
// iterations"; DESIGN.md section 5.1 on how the group size trades L2 residency against
// the distance between dependent products), and the products inside a group are ordered
// iteration -> op -> submatrix -> tile  so that by the time a CTA reaches a tile of op s of a submatrix,
// op s-1 of that submatrix finished several waves ago.  CTAs claim tile indices in that order with one
// atomicAdd per tile.  The dependency itself is enforced by a per-submatrix counter in global memory
// (ready[m] = ops completed, acquire/release at GPU scope), not by a grid barrier; a tile only ever
// waits for tiles with a smaller index, all of which have been claimed by running CTAs, and all CTAs
// are co-resident (cooperative launch), so the schedule cannot deadlock.
//
// Layout facts:
//   * all matrices are column-major, so the A operand (M x K) is M-major and the B operand (K x N) is
//     K-major in shared memory; one TMA tensor map per FP16 buffer with box {64 storage rows,
//     64 storage columns} serves both roles (A: 2 boxes per 128-row tile and K block; B: one box per
//     64 tile columns), 128-byte swizzle.
//   * accumulator: 128 TMEM lanes = tile rows, one 32-bit column per tile column; two accumulator
//     stages so the epilogue of tile i overlaps the MMAs of tile i+1.
//   * the FP32 master iterate (reading 12) is read in the epilogue with L2-only loads
//     (ld.global.cg: other SMs wrote it) issued one chunk ahead, and written back with coalesced stores.
//
// Warp roles (352 threads): warp 0 = scheduler (claims the next tiles and resolves their dependencies, up
// to kRing tiles ahead), warp 1 = MMA issuer (whole warp, one elected lane issues; + TMEM allocation),
// warp 2 = TMA producer, warps 3..10 =
// epilogue (TMEM lane quadrant = warp_id % 4; the two warps of a quadrant take alternate 32-column
// chunks of the tile).
#include "common.cuh"
#include "chain_epilogue.cuh"

namespace {

constexpr int kThreads = 352;
constexpr int kEpiWarps = 8;
constexpr int kBK = 64;                  // K elements per pipeline stage (= one 128-byte swizzle row)
constexpr int kMaxStages = 8;
constexpr int kTmemCols = 512;
constexpr int kBoxBytes = 64 * 128;      // one {64 x 64} FP16 box
constexpr int kATileBytes = 2 * kBoxBytes;
constexpr int kRing = 2;                 // tile-command ring depth (how far the scheduler claims ahead)
constexpr int kSmemLimit = 232448 - 2048;  // 227 KB minus the static part (barriers, commands)
constexpr int32_t kDone = 0x7fffffff;

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra WAIT_DONE;\n\t"
      "bra WAIT_LOOP;\n\t"
      "WAIT_DONE:\n\t"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0,
                                            int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, "
      "%4, %5}], [%2];" ::"r"(smem_u32(dst)),
      "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
// one lane of the (converged) warp; the compiler keeps code guarded by it on the uniform datapath
__device__ __forceinline__ bool elect_one() {
  uint32_t p;
  asm volatile(
      "{\n\t"
      ".reg .pred P;\n\t"
      "elect.sync _|P, 0xffffffff;\n\t"
      "selp.u32 %0, 1, 0, P;\n\t"
      "}\n"
      : "=r"(p));
  return p != 0;
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(
                   smem_u32(bar))
               : "memory");
}
// Same with the descriptors given as 32-bit halves: the high half (stride offset, version, swizzle) is a
// constant, the low half is base + k * step, so the single issuing thread spends a handful of integer
// instructions per MMA instead of rebuilding two 64-bit descriptors (it was issue-bound at ~200 cycles
// per MMA against the 128 the tensor pipe needs, profiles/r1_k_chain_sign_w32768.md).
__device__ __forceinline__ void tc_mma_f16_lh(uint32_t tmem_d, uint32_t a_lo, uint32_t b_lo, uint32_t desc_hi,
                                              uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      ".reg .b64 da, db;\n\t"
      "setp.ne.b32 p, %5, 0;\n\t"
      "mov.b64 da, {%1, %3};\n\t"
      "mov.b64 db, {%2, %3};\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %4, p;\n\t"
      "}\n" ::"r"(tmem_d),
      "r"(a_lo), "r"(b_lo), "r"(desc_hi), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ int32_t ld_acquire(const int32_t *p) {
  int32_t v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
#ifdef NOLSM_TRACE
__device__ long long g_trace[4][4096][2];
#define TRACE(role, ti, j) do { if (blockIdx.x == 0 && (ti) < 4096) g_trace[role][ti][j] = clock64(); } while (0)
#define TRACEV(role, ti, j, v) do { if (blockIdx.x == 0 && (ti) < 4096) g_trace[role][ti][j] = (v); } while (0)
__device__ long long g_trace2[4096][8];
__device__ long long g_wait[4096][4];
#define TRACE2(ti, j) do { if (blockIdx.x == 0 && warp == 3 && lane == 0 && (ti) < 4096) g_trace2[ti][j] = clock64(); } while (0)
#else
#define TRACE2(ti, j)
#define TRACE(role, ti, j)
#define TRACEV(role, ti, j, v)
#endif

using chainep::TileCmd;
using chainep::ChainArgs;

__global__ void __launch_bounds__(kThreads, 1) k_chain(const ChainArgs args) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ uint64_t full_bar[kMaxStages], empty_bar[kMaxStages], tfull_bar[2], tempty_bar[2];
  __shared__ uint64_t cmd_full[kRing], cmd_empty[kRing];
  __shared__ TileCmd cmds[kRing];
  __shared__ uint32_t tmem_base_s;

  const ChainProgram &pg = args.prog;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  // stage layout: [A hi 16K][B hi b_bytes][A lo 16K][B lo b_bytes]
  const int off_b = kATileBytes, off_a_lo = kATileBytes + args.b_bytes, off_b_lo = 2 * kATileBytes + args.b_bytes;

  if (threadIdx.x == 0) {
    for (int s = 0; s < args.stages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(&tfull_bar[a], 1); mbar_init(&tempty_bar[a], kEpiWarps); }
    for (int r = 0; r < kRing; ++r) { mbar_init(&cmd_full[r], 1); mbar_init(&cmd_empty[r], 2 + kEpiWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                 "r"(kTmemCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;

  if (warp == 0) {
    // ===================== scheduler =====================
    if (lane == 0) {
      int slot = 0;
      uint32_t ring_phase = 0;
      const int T = args.mt * args.ntl;
      const int limit = pg.fixed_iter > 0 ? min(pg.fixed_iter, pg.max_iter) : pg.max_iter;
      const int n_groups = (args.count + pg.group - 1) / pg.group;
      // Dynamic, in-order tile claims: a tile only depends on tiles with a smaller index, all of which
      // have been claimed by running CTAs, so the schedule cannot deadlock and balances itself.
      const int64_t per_group = (int64_t)limit * pg.n_ops * pg.group * T;   // index space of one (full) group
      int g_checked = -1, k_checked = 0;
      for (;;) {
        const int64_t L = (int64_t)atomicAdd(args.tile_counter, 1ull);
        const int g = (int)(L / per_group);
        if (g >= n_groups) break;
        const int64_t Lg = L - (int64_t)g * per_group;
        const int gbase = g * pg.group;
        const int gs = min(pg.group, args.count - gbase);
        const int per_seg = gs * T;
        if (Lg >= (int64_t)limit * pg.n_ops * per_seg) continue;   // index padding of the last group
        const int seg = (int)(Lg / per_seg), rem = (int)(Lg % per_seg);
        const int k = seg / pg.n_ops, op = seg % pg.n_ops;
        if (g != g_checked) { g_checked = g; k_checked = 0; }
        if (k != k_checked) {   // whole group converged: move the claim counter past it
          if (ld_acquire(&args.group_active[g]) == 0) {
            atomicMax(args.tile_counter, (unsigned long long)((int64_t)(g + 1) * per_group));
            continue;
          }
          k_checked = k;
        }
        const int ml = rem / T, t = rem % T;
        const int m = gbase + ml;
        const int n = args.dims[m];
        const int n16 = (n + 15) & ~15;
        const int m0 = (t % args.mt) * NOLSM_TILE_M, n0 = (t / args.mt) * args.bn;
        if (m0 >= n || n0 >= n16) continue;          // tile outside this submatrix
        const int need = k * pg.n_ops + op;          // ops of this submatrix that must be complete
        if (need > 0) {
          int32_t r = ld_acquire(&args.ready[m]);
          while (r < need) { __nanosleep(64); r = ld_acquire(&args.ready[m]); }
          if (r == kDone) continue;                  // submatrix finished at an earlier iteration
        }
        const int kblocks = (n16 + kBK - 1) / kBK;
        {
          mbar_wait(&cmd_empty[slot], ring_phase ^ 1u);
          cmds[slot] = TileCmd{m, m0, n0, min(args.bn, n16 - n0), kblocks, (n16 - (kblocks - 1) * kBK) / 16, op,
                                  k | (pg.parity_from_iters ? (((args.iters[m] + 1) & 1) << 30) : 0)};
          mbar_arrive(&cmd_full[slot]);
          if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
        }
      }
      mbar_wait(&cmd_empty[slot], ring_phase ^ 1u);
      cmds[slot] = TileCmd{0, 0, 0, 0, 0, 0, -1, 0};
      mbar_arrive(&cmd_full[slot]);
    }
  } else if (warp == 2) {
    // ===================== TMA producer =====================
    if (lane == 0) {
#ifdef NOLSM_NOTMA
      int tma_issued = 0;
#endif
#ifdef NOLSM_TRACE
      int tti = 0;
#endif
      int stage = 0, slot = 0;
      uint32_t phase = 0, ring_phase = 0;
      for (;;) {
        mbar_wait(&cmd_full[slot], ring_phase);
        const TileCmd c = cmds[slot];
        mbar_arrive(&cmd_empty[slot]);
        if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
        if (c.op < 0) break;
        TRACE(2, tti, 0);
        fence_proxy_async();   // other CTAs' generic-proxy writes (ordered by the scheduler's acquire) -> TMA reads
        const ChainOp &o = pg.ops[c.op];
        const int par = chainep::cmd_par(c);
        const int m = c.mat, m0 = c.m0, n0 = c.n0;
        const bool split = o.a_lo[par] >= 0;
        const int nbox = (c.nt + 63) >> 6;
        const uint32_t bytes = (uint32_t)(kATileBytes + nbox * kBoxBytes) * (split ? 2u : 1u);
        const CUtensorMap *ma = &args.maps[o.a[par]], *mb = &args.maps[o.b[par]];
        const CUtensorMap *mal = split ? &args.maps[o.a_lo[par]] : nullptr;
        const CUtensorMap *mbl = split ? &args.maps[o.b_lo[par]] : nullptr;
        for (int kb = 0; kb < c.kblocks; ++kb) {
          mbar_wait(&empty_bar[stage], phase ^ 1u);
          uint8_t *st = smem + (size_t)stage * args.stage_bytes;
#ifdef NOLSM_NOTMA   // timing experiment only: the barrier protocol without any operand traffic (results are wrong)
          if (tma_issued >= args.stages) { mbar_arrive(&full_bar[stage]); if (++stage == args.stages) { stage = 0; phase ^= 1u; } continue; }
          ++tma_issued;
#endif
          mbar_expect_tx(&full_bar[stage], bytes);
          const int k0 = kb * kBK;
          tma_load_3d(st, ma, &full_bar[stage], m0, k0, m);
          tma_load_3d(st + kBoxBytes, ma, &full_bar[stage], m0 + 64, k0, m);
          for (int j = 0; j < nbox; ++j)
            tma_load_3d(st + off_b + j * kBoxBytes, mb, &full_bar[stage], k0, n0 + 64 * j, m);
          if (split) {
            tma_load_3d(st + off_a_lo, mal, &full_bar[stage], m0, k0, m);
            tma_load_3d(st + off_a_lo + kBoxBytes, mal, &full_bar[stage], m0 + 64, k0, m);
            for (int j = 0; j < nbox; ++j)
              tma_load_3d(st + off_b_lo + j * kBoxBytes, mbl, &full_bar[stage], k0, n0 + 64 * j, m);
          }
          if (++stage == args.stages) { stage = 0; phase ^= 1u; }
        }
        TRACE(2, tti, 1);
#ifdef NOLSM_TRACE
        ++tti;
#endif
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    // The whole warp walks the tile sequence (uniform control flow, operands in uniform registers); one
    // elected lane issues the MMAs, commits and arrivals.
    {
      const bool one = elect_one();
#ifdef NOLSM_TRACE
      int mti = 0;
#endif
      int stage = 0, slot = 0, acc = 0;
      uint32_t phase = 0, ring_phase = 0, acc_phase = 0;
      const uint32_t smem_base = smem_u32(smem);
      // high half of every operand descriptor: stride offset 1024 B (8-row atoms), version 1, 128-byte swizzle
      constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);
      for (;;) {
        mbar_wait(&cmd_full[slot], ring_phase);
        const TileCmd c = cmds[slot];
        __syncwarp();
        if (one) mbar_arrive(&cmd_empty[slot]);
        if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
        if (c.op < 0) break;
        const bool split = pg.ops[c.op].a_lo[chainep::cmd_par(c)] >= 0;
        // instruction descriptor: D=F32, A=B=F16, A M-major, B K-major, N = nt, M = 128
        const uint32_t idesc = (1u << 4) | (1u << 15) | ((uint32_t)(c.nt >> 3) << 17) | ((128u >> 4) << 24);
        TRACE(0, mti, 0);
        mbar_wait(&tempty_bar[acc], acc_phase ^ 1u);
        tc_fence_after();
        TRACE(0, mti, 1);
#ifdef NOLSM_TRACE
        ++mti;
#endif
        const uint32_t d_main = tmem_base + (uint32_t)(acc * 256);
        const uint32_t d_corr = d_main + 128;
#ifdef NOLSM_TRACE
        long long wsum = 0, t_begin = clock64();
#endif
        for (int kb = 0; kb < c.kblocks; ++kb) {
#ifdef NOLSM_TRACE
          long long w0 = clock64();
#endif
          mbar_wait(&full_bar[stage], phase);
#ifdef NOLSM_TRACE
          wsum += clock64() - w0;
#endif
          tc_fence_after();
          // descriptor low halves: (address >> 4) | leading offset << 16; A (M-major): leading offset = the
          // second 64-row chunk (8192 B), +2048 B per K=16 step; B (K-major): leading offset 16 B, +32 B per step
          const uint32_t sa = smem_base + (uint32_t)stage * (uint32_t)args.stage_bytes;
          const uint32_t a_lo = ((sa >> 4) & 0x3FFFu) | ((uint32_t)(kBoxBytes >> 4) << 16);
          const uint32_t b_lo = (((sa + off_b) >> 4) & 0x3FFFu) | (1u << 16);
          const int steps = kb == c.kblocks - 1 ? c.ktail : kBK / 16;
          if (one) {
          if (!split) {
            tc_mma_f16_lh(d_main, a_lo, b_lo, kDescHi, idesc, kb ? 1u : 0u);
            if (steps > 1) tc_mma_f16_lh(d_main, a_lo + 128u, b_lo + 2u, kDescHi, idesc, 1u);
            if (steps > 2) tc_mma_f16_lh(d_main, a_lo + 256u, b_lo + 4u, kDescHi, idesc, 1u);
            if (steps > 3) tc_mma_f16_lh(d_main, a_lo + 384u, b_lo + 6u, kDescHi, idesc, 1u);
          } else {
            const uint32_t al_lo = (((sa + off_a_lo) >> 4) & 0x3FFFu) | ((uint32_t)(kBoxBytes >> 4) << 16);
            const uint32_t bl_lo = (((sa + off_b_lo) >> 4) & 0x3FFFu) | (1u << 16);
            for (int k4 = 0; k4 < steps; ++k4) {
              const uint32_t accum = (kb | k4) ? 1u : 0u;
              tc_mma_f16_lh(d_main, a_lo + 128u * k4, b_lo + 2u * k4, kDescHi, idesc, accum);
              tc_mma_f16_lh(d_corr, a_lo + 128u * k4, bl_lo + 2u * k4, kDescHi, idesc, accum);
              tc_mma_f16_lh(d_corr, al_lo + 128u * k4, b_lo + 2u * k4, kDescHi, idesc, 1u);
            }
          }
          tc_commit(&empty_bar[stage]);
          }
          __syncwarp();
          if (++stage == args.stages) { stage = 0; phase ^= 1u; }
        }
        if (one) tc_commit(&tfull_bar[acc]);
        __syncwarp();
#ifdef NOLSM_TRACE
        if (blockIdx.x == 0 && mti - 1 < 4096) { g_wait[mti - 1][0] = wsum; g_wait[mti - 1][2] = clock64() - t_begin; }
#endif
        if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      }
    }
  } else {
    // ===================== epilogue =====================
    const int q = warp & 3;          // TMEM lane quadrant this warp may access
#ifdef NOLSM_TRACE
    int eti = 0;
#endif
    const int chunk_first = (warp - 3) >> 2;   // this warp's chunks: chunk_first, chunk_first + 2, ...
    int slot = 0, acc = 0, tile_seq = 0;
    uint32_t ring_phase = 0, acc_phase = 0;
    for (;;) {
      mbar_wait(&cmd_full[slot], ring_phase);
      const TileCmd c = cmds[slot];
      __syncwarp();
      if (lane == 0) mbar_arrive(&cmd_empty[slot]);
      if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
      if (c.op < 0) break;
      chainep::EpiTile t;
      chainep::epi_begin(args, c, c.m0 + q * 32, true, lane, chunk_first, t);
      if (warp == 3 && lane == 0) { TRACE(1, eti, 0); }
      mbar_wait(&tfull_bar[acc], acc_phase);
      tc_fence_after();
      if (warp == 3 && lane == 0) { TRACE(1, eti, 1); TRACEV(3, eti, 0, (long long)c.op); }
      const uint32_t t_main = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * 256);
#ifdef NOLSM_TRACE
      float ss = chainep::epi_chunks(args, c, t, t_main, lane,
                                     (blockIdx.x == 0 && warp == 3 && eti < 4096) ? g_trace2[eti] : nullptr);
#else
      float ss = chainep::epi_chunks(args, c, t, t_main, lane);
#endif
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tempty_bar[acc]);
      if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      if (t.o->resid) {
        for (int d = 16; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
        if (lane == 0) atomicAdd(&args.resid2[(size_t)(chainep::cmd_iter(c) % NOLSM_MAX_RESID_SLOTS) * args.count + c.mat], ss);
      }
      TRACE2(eti, 5);
      // all epilogue warps have issued their stores and residual atomics: one thread publishes the tile
      asm volatile("bar.sync 1, %0;" ::"n"(kEpiWarps * 32) : "memory");
      if (warp - 3 == (tile_seq & (kEpiWarps - 1)) && lane == 0)
        chainep::epi_complete<NOLSM_TILE_M, 16, 1>(args, c);
      ++tile_seq;
      if (warp == 3 && lane == 0) { TRACE(3, eti, 1); }
#ifdef NOLSM_TRACE
      ++eti;
#endif
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols) : "memory");
  }
}

// Reset of the per-launch control state.
__global__ void __launch_bounds__(256)
k_chain_reset(int count, int group, int32_t *ready, int32_t *tiles_done, int32_t *state, int32_t *group_active,
              unsigned long long *tile_counter, float *resid2, int resid_elems, int32_t *iters, float *lastres,
              int touch_stats) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) *tile_counter = 0ull;
  const int stride = gridDim.x * blockDim.x;
  for (int m = i; m < count; m += stride) {
    ready[m] = 0;
    tiles_done[m] = 0;
    state[m] = 0x7fffffff;
    if (touch_stats) { iters[m] = 0; lastres[m] = -1.f; }
  }
  const int n_groups = (count + group - 1) / group;
  for (int g = i; g < n_groups; g += stride) group_active[g] = min(group, count - g * group);
  for (int e = i; e < resid_elems; e += stride) resid2[e] = 0.f;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

// stored matrix: dim0 = row index (contiguous), dim1 = column index, dim2 = submatrix
// FP16 operand buffer: {64 storage rows, 64 storage columns} box with 128-byte swizzle, one map serving
// both operand roles (see the header comment)
nolsm_status encode_map(nolsm_ctx *ctx, CUtensorMap *map, void *ptr, int ld, int count) {
  cuuint64_t dims[3] = {(cuuint64_t)ld, (cuuint64_t)ld, (cuuint64_t)count};
  cuuint64_t strides[2] = {(cuuint64_t)ld * sizeof(__half), (cuuint64_t)ld * ld * sizeof(__half)};
  cuuint32_t box[3] = {64u, 64u, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = reinterpret_cast<EncodeTiledFn>(ctx->encode_tiled)(
      map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, ptr, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
      CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    ctx->err = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r);
    return NOLSM_ECUDA;
  }
  return NOLSM_OK;
}

}  // namespace

#ifdef NOLSM_TRACE
extern "C" void nolsm_debug_trace(long long *host_out) {
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(host_out, g_trace, sizeof(g_trace));
}
extern "C" void nolsm_debug_pwait1(long long *host_out) { cudaMemcpyFromSymbol(host_out, g_wait, sizeof(g_wait)); }
extern "C" void nolsm_debug_trace2(long long *host_out) { cudaMemcpyFromSymbol(host_out, g_trace2, sizeof(g_trace2)); }
#endif

nolsm_status umma_init(nolsm_ctx *ctx) {
  ctx->umma_ok = false;
  cudaDriverEntryPointQueryResult qres;
  void *fn = nullptr;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || fn == nullptr || qres != cudaDriverEntryPointSuccess) {
    ctx->err = "cuTensorMapEncodeTiled entry point not available";
    cudaGetLastError();
    return NOLSM_ECUDA;
  }
  ctx->encode_tiled = fn;
  e = cudaFuncSetAttribute(k_chain, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit);
  if (e != cudaSuccess) {
    ctx->err = std::string("cudaFuncSetAttribute(k_chain): ") + cudaGetErrorString(e);
    cudaGetLastError();
    return NOLSM_ECUDA;
  }
  int coop = 0;
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device);
  if (!coop) {
    ctx->err = "device does not support cooperative launches";
    return NOLSM_ECUDA;
  }
  ctx->umma_ok = true;
  pair_init(ctx);   // optional: the single-CTA engine is the fallback
  mcast_init(ctx);
  return NOLSM_OK;
}

nolsm_status umma_make_maps(nolsm_ctx *ctx, nolsm_batch *b) {
  b->maps_valid = false;
  if (!ctx->umma_ok || b->count == 0) return NOLSM_OK;
  std::vector<CUtensorMap> maps(b->n_half);
  for (int i = 0; i < b->n_half; ++i) {
    nolsm_status s = encode_map(ctx, &maps[i], b->h[i], b->ld, b->count);
    if (s != NOLSM_OK) return s;
  }
  if (!b->d_maps) {
    if (cudaMalloc(&b->d_maps, sizeof(CUtensorMap) * NOLSM_MAX_HALF) != cudaSuccess) {
      cudaGetLastError();
      ctx->err = "cudaMalloc of the tensor maps failed";
      return NOLSM_ENOMEM;
    }
  }
  NOLSM_CUDA(ctx, cudaMemcpy(b->d_maps, maps.data(), sizeof(CUtensorMap) * maps.size(), cudaMemcpyHostToDevice));
  b->maps_valid = true;
  return NOLSM_OK;
}

// Runs `prog` over every submatrix of the batch.  touch_stats: reset and fill iters / lastres.
cudaError_t launch_chain(nolsm_ctx *ctx, const nolsm_batch *b, const ChainProgram &prog, const float *alpha_div,
                         bool touch_stats, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  if (!ctx->umma_ok || !b->maps_valid) return cudaErrorNotSupported;
  ChainArgs a;
  memset(&a, 0, sizeof(a));
  a.prog = prog;
  bool split = false;
  for (int i = 0; i < prog.n_ops; ++i) split |= prog.ops[i].a_lo[0] >= 0 || prog.ops[i].a_lo[1] >= 0;
  const int n16max = (b->max_n + 15) & ~15;
  a.bn = std::min(split ? 128 : 256, n16max);
  a.b_bytes = ((a.bn + 63) / 64) * kBoxBytes;
  a.stage_bytes = (kATileBytes + a.b_bytes) * (split ? 2 : 1);
  a.stages = std::min(kMaxStages, (kSmemLimit - 1024) / a.stage_bytes);
  a.mt = (b->max_n + NOLSM_TILE_M - 1) / NOLSM_TILE_M;
  a.ntl = (n16max + a.bn - 1) / a.bn;
  a.maps = b->d_maps;
  a.n_half = b->n_half;
  a.n_unit = b->n_unit;
  for (int i = 0; i < b->n_half; ++i) a.hbuf[i] = b->h[i];
  for (int i = 0; i < b->n_unit; ++i) a.ubuf[i] = b->u[i];
  a.count = b->count;
  a.ld = b->ld;
  a.slab = (int64_t)b->ld * b->ld;
  a.dims = b->d_dims;
  a.alpha_div = alpha_div;
  a.ready = b->d_ready;
  a.tiles_done = b->d_tiles_done;
  a.state = b->d_state;
  a.iters = b->d_iters;
  a.alpha_tab = prog.use_alpha_tab ? b->d_alpha : nullptr;
  a.group_active = b->d_group_active;
  a.tile_counter = b->d_tile_counter;
  a.resid2 = b->d_resid2;
  a.lastres = b->d_lastres;
  if (a.prog.group <= 0) a.prog.group = 1;
  const int slots = std::min(prog.max_iter, NOLSM_MAX_RESID_SLOTS);
  k_chain_reset<<<64, 256, 0, st>>>(b->count, a.prog.group, a.ready, a.tiles_done, a.state, a.group_active,
                                    a.tile_counter, a.resid2, slots * b->count, a.iters, a.lastres, touch_stats ? 1 : 0);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const int forced = ctx->cfg.flags & (NOLSM_FLAG_PAIR | NOLSM_FLAG_MCAST | NOLSM_FLAG_SINGLE);
  if (ctx->pair_ok && ((forced & NOLSM_FLAG_PAIR) || (forced == 0 && b->prefer_pair)))
    return launch_chain_pair(ctx, b, a.prog, alpha_div, st);
  if (ctx->mcast_ok && (ctx->cfg.flags & NOLSM_FLAG_MCAST)) return launch_chain_mcast(ctx, b, a.prog, alpha_div, st);
  const int smem_bytes = a.stages * a.stage_bytes + 1024;
  void *params[] = {&a};
  return cudaLaunchCooperativeKernel(reinterpret_cast<void *>(k_chain), dim3(ctx->sm_count), dim3(kThreads), params,
                                     (size_t)smem_bytes, st);
}
