// The batched matrix-iteration engine: ONE persistent, cooperative kernel runs a whole chain of
// dependent n x n x n products (every iteration of Eq. 9-10, or of Eq. 15-17
// PAPER.md:203-215) for every submatrix of a batch on the 5th-generation tensor cores
// (tcgen05 + TMEM + TMA), sm_100a only.  Two instantiations of one kernel template:
//   k_chain<false, *>  one CTA per tile of N rows x 128 columns of the result (tcgen05.mma.cta_group::1)
//   k_chain<true, *>   two CTAs of a cluster (one TPC) per tile of N rows x 256 columns (cta_group::2): each CTA stages
//                   its own 128 columns of the right operand and only HALF of the rows of the left operand, so the
//                   operand bytes an SM takes in per 64-deep K block drop from 48 KB to 32 KB.
//
// Why one kernel: the two products of a sign iteration are strictly dependent and one product of an
// n ~ 860 submatrix is < 1 us of the whole GPU, so kernel boundaries would cost more than the work, and
// a batch-wide launch per product streams every iterate through HBM (18 n^2 bytes per 4 n^3 FLOP,
// DESIGN.md "Roofline").
//
// Schedule: a ROLLING WINDOW of W submatrices (the B200 analogue of the paper's "caching strategy for the
// matrices during the iterations").  Window slot s holds one submatrix and the index of its next
// product; the work is enumerated as  round -> slot -> tile : in every round each slot contributes the tiles of
// ONE product of its submatrix, so consecutive (dependent) products of a submatrix are W - 1 other products apart
// and the iterates of the W submatrices stay in L2 from the first to the last iteration.  A submatrix that
// converges leaves its slot to the next submatrix of the batch, so the window never drains between groups.
// CTAs claim tile indices in that order with one atomicAdd per tile.  The dependency itself is enforced by the
// slot's state word in global memory (round | product index | submatrix, acquire/release at GPU scope), not by a
// grid barrier: a tile of round r of slot s waits until the slot has completed round r - 1; it only ever waits for
// tiles with a smaller index, all of which have been claimed by running CTAs, and all CTAs are co-resident
// (cooperative launch), so the schedule cannot deadlock.
//
// Layout facts:
//   * all matrices are column-major.  The tensor cores compute the TRANSPOSED product C^T = R^T L^T of every
//     C = L R: the MMA's M side runs over 128 COLUMNS of C and takes the right operand R (for a fixed column
//     its K elements are contiguous: K-major), the N side runs over up to 256 ROWS of C and takes the left
//     operand L (for a fixed k its rows are contiguous: MN-major).  Nothing is transposed in memory; one TMA
//     tensor map per FP16 buffer with box {64 storage rows, 64 storage columns}, 128-byte swizzle, serves both
//     roles.  The point is the epilogue: TMEM lane = column of C, TMEM column = row of C, so a thread holds 32
//     CONSECUTIVE elements of a column and moves them with 16-byte accesses (chain_epilogue.cuh).
//   * accumulator: 128 TMEM lanes = tile columns, one 32-bit TMEM column per tile row; two accumulator
//     stages so the epilogue of tile i overlaps the MMAs of tile i+1.
//
// Warp roles (384 threads): warp 0 = scheduler (leader CTA; claims the next tile, resolves its dependency and
// writes the tile command into the ring of every CTA of the cluster), warp 1 = MMA issuer (leader CTA; whole warp,
// one elected lane issues; + TMEM allocation), warp 2 = TMA producer of the operands, warp 3 = epilogue agent (one
// thread: TMA loads of the FP16 add-in into the staging buffers, TMA stores of the FP16 results out of them,
// publication of the tile; chain_epilogue.cuh), warps 4..11 = epilogue compute (TMEM lane quadrant = warp_id % 4;
// the two warps of a quadrant take the two 32-row halves of the 64-row chunks of the tile).
#include "common.cuh"
#include "chain_epilogue.cuh"

namespace {

constexpr int kEpiWarps = chainep::kComputeWarps;
constexpr int kAgentWarp = 3;
constexpr int kFirstEpiWarp = 4;
constexpr int kThreads = 32 * (kFirstEpiWarp + kEpiWarps);
constexpr int kBK = 64;                  // K elements per pipeline stage (= one 128-byte swizzle row)
constexpr int kMaxStages = 8;
constexpr int kTmemCols = 512;
constexpr int kBoxBytes = 64 * 128;      // one {64 x 64} FP16 box
constexpr int kATileBytes = 2 * kBoxBytes;   // this CTA's 128 rows x 64 K
constexpr int kRing = 2;                 // tile-command ring depth
constexpr int kClaimLead = 4;            // the next tile is claimed when the producer is this many K blocks from the
                                         // end of the current one: late enough to keep dependent products close,
                                         // early enough to hide the claim's atomic + acquire round trips
constexpr int kSmemLimit = 232448 - 2048;  // 227 KB minus the static part (barriers, commands)

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
// shared::cluster address of the same variable in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(uint32_t saddr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
  return r;
}
__device__ __forceinline__ uint32_t cluster_rank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
// arrive on a barrier of CTA `rank` of the cluster (kPair) or of this CTA
template <bool kPair>
__device__ __forceinline__ void mbar_arrive(uint64_t *bar, uint32_t rank = 0) {
  if constexpr (kPair)
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(mapa(smem_u32(bar), rank))
                 : "memory");
  else
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// wait; with acquire at cluster scope when the arrivals may come from the peer CTA
template <bool kPair>
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  if constexpr (kPair)
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "PWAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra PWAIT_DONE;\n\t"
        "bra PWAIT_LOOP;\n\t"
        "PWAIT_DONE:\n\t"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
  else
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
// one non-blocking probe of a barrier phase
template <bool kPair>
__device__ __forceinline__ bool mbar_test(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  if constexpr (kPair)
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.test_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  else
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  return ok != 0;
}
// TMA load into THIS CTA's shared memory; kPair: the bytes are counted on the LEADER's barrier
template <bool kPair>
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1,
                                            int c2) {
  if constexpr (kPair)
    asm volatile(
        "cp.async.bulk.tensor.3d.cta_group::2.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, "
        "{%3, %4, %5}], [%2];" ::"r"(smem_u32(dst)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(mapa(smem_u32(bar), 0)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
  else
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
// arrives on the barrier (kPair: at the same offset in BOTH CTAs) once all prior MMAs of this thread are done
template <bool kPair>
__device__ __forceinline__ void tc_commit(uint64_t *bar) {
  if constexpr (kPair)
    asm volatile(
        "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
            smem_u32(bar)),
        "h"((uint16_t)3)
        : "memory");
  else
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
// The operand descriptors are given as 32-bit halves: the high half (stride offset, version, swizzle) is a
// constant, the low half is base + k * step, so the single issuing thread spends a handful of integer
// instructions per MMA instead of rebuilding two 64-bit descriptors (it was issue-bound at ~200 cycles
// per MMA against the 128 the tensor pipe needs, profiles/r1_k_chain_sign_w32768.md).
template <bool kPair>
__device__ __forceinline__ void tc_mma(uint32_t tmem_d, uint32_t a_lo, uint32_t b_lo, uint32_t desc_hi, uint32_t idesc,
                                       uint32_t accumulate) {
  if constexpr (kPair)
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        ".reg .b64 da, db;\n\t"
        "setp.ne.b32 p, %5, 0;\n\t"
        "mov.b64 da, {%1, %3};\n\t"
        "mov.b64 db, {%2, %3};\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], da, db, %4, p;\n\t"
        "}\n" ::"r"(tmem_d),
        "r"(a_lo), "r"(b_lo), "r"(desc_hi), "r"(idesc), "r"(accumulate)
        : "memory");
  else
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
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ int32_t ld_acquire(const int32_t *p) {
  int32_t v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

using chainep::TileCmd;
using chainep::ChainArgs;

// kFeat: feature bits of chain_epilogue.cuh (kFeat*); launch_chain picks the smallest instantiation that covers a program
template <bool kPair, int kFeat>
__global__ void __launch_bounds__(kThreads, 1) k_chain(const ChainArgs args) {
  constexpr int kCtas = kPair ? 2 : 1;
  constexpr int kTileM = NOLSM_TILE_M * kCtas;      // rows of a tile
  constexpr int kColRound = kPair ? 32 : 16;        // tile columns are multiples of this
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ uint64_t full_bar[kMaxStages], empty_bar[kMaxStages], tfull_bar[2], tempty_bar[2];
  __shared__ uint64_t cmd_full[kRing], cmd_empty[kRing], claim_go;
  __shared__ __align__(16) TileCmd cmds[kRing];
  __shared__ chainep::EpiBars ebars;
  __shared__ uint32_t tmem_base_s;

  const ChainProgram &pg = args.prog;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long t_start = clock64();
  const uint32_t rank = kPair ? cluster_rank() : 0u;
  const bool leader = rank == 0;
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  // stage layout: [A hi 16K][B hi b_bytes][A lo 16K][B lo b_bytes]
  // a stage: [M-side hi][N-side hi][N-side lo][M-side lo] -- the lo boxes of the N side directly behind its hi boxes
  const int off_b = kATileBytes, off_b_lo = kATileBytes + args.b_bytes, off_a_lo = kATileBytes + 2 * args.b_bytes;
  uint8_t *staging = smem + (size_t)args.stages * args.stage_bytes;   // epilogue staging buffers behind the operand ring

  if (threadIdx.x == 0) {
    // `full` (operands landed) and `tmem empty` are waited on in the leader: both CTAs' TMA loads signal the
    // leader's `full` barrier, the peer's epilogue warps arrive remotely on `tmem empty`
    for (int s = 0; s < args.stages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(&tfull_bar[a], 1); mbar_init(&tempty_bar[a], kCtas * kEpiWarps); }
    // command ring: filled by the leader's scheduler in every CTA; freed (leader's barrier) by the leader's
    // MMA issuer + every CTA's TMA producer and epilogue warps
    // MMA issuer + every CTA's TMA producer, epilogue compute warps and epilogue agents
    for (int r = 0; r < kRing; ++r) { mbar_init(&cmd_full[r], 1); mbar_init(&cmd_empty[r], 1 + kCtas * (1 + kEpiWarps + 1)); }
    mbar_init(&claim_go, 1);
    for (int b = 0; b < 2; ++b) { mbar_init(&ebars.in_full[b], 1); mbar_init(&ebars.out_ready[b], kEpiWarps); }
    mbar_init(&ebars.tile_done[0], kEpiWarps);
    mbar_init(&ebars.tile_done[1], kEpiWarps);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    if constexpr (kPair) {
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                   "r"(kTmemCols)
                   : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                   "r"(kTmemCols)
                   : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
  }
  tc_fence_before();
  __syncthreads();
  if constexpr (kPair) cluster_sync();   // barriers of both CTAs initialised before any remote arrive / multicast commit
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;

  if (warp == 0) {
    // ===================== scheduler (leader CTA) =====================
    if (leader && lane == 0) {
      int slot = 0;
      uint32_t ring_phase = 0, go_phase = 0;
      bool gate = false;      // a command has been handed to the producer: wait for its `claim_go` before claiming again
      const int T = args.mt * args.ntl;
      const int W = args.window;
      const int64_t per_round = (int64_t)W * T;
      auto push = [&](const TileCmd &cmd) {
        mbar_wait<kPair>(&cmd_empty[slot], ring_phase ^ 1u);
        cmds[slot] = cmd;
        if constexpr (kPair) {
          const uint32_t remote = mapa(smem_u32(&cmds[slot]), 1);
          asm volatile("st.shared::cluster.v4.s32 [%0], {%1, %2, %3, %4};" ::"r"(remote), "r"(cmd.mat), "r"(cmd.m0),
                       "r"(cmd.n0), "r"(cmd.nt)
                       : "memory");
          asm volatile("st.shared::cluster.v4.s32 [%0], {%1, %2, %3, %4};" ::"r"(remote + 16), "r"(cmd.kblocks),
                       "r"(cmd.ktail), "r"(cmd.op), "r"(cmd.iter)
                       : "memory");
          asm volatile("st.shared::cluster.v4.s32 [%0], {%1, %2, %3, %4};" ::"r"(remote + 32), "r"(cmd.slot), "r"(0),
                       "r"(0), "r"(0)
                       : "memory");
          mbar_arrive<true>(&cmd_full[slot], 0);
          mbar_arrive<true>(&cmd_full[slot], 1);
        } else {
          mbar_arrive<false>(&cmd_full[slot]);
        }
        if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
      };
      for (;;) {
        if (gate) { mbar_wait<false>(&claim_go, go_phase); go_phase ^= 1u; gate = false; }
        const int64_t L = (int64_t)atomicAdd(args.tile_counter, 1ull);
        const uint32_t round = (uint32_t)(L / per_round);
        const int rem = (int)(L % per_round);
        const int s = rem / T, t = rem % T;
        // the slot must have completed round - 1 (or be retired); a tile only waits for smaller tile indices
        unsigned long long st = ld_acquire_u64(&args.slot_state[s]);
        while (chainep::slot_round(st) < round) { __nanosleep(64); st = ld_acquire_u64(&args.slot_state[s]); }
        if (st == chainep::kSlotDead) {
          if (ld_acquire(&args.sched[1]) >= W) break;   // every slot retired: the batch is done
          continue;
        }
        if (chainep::slot_round(st) != round) continue;  // the round went by without this tile: it lies outside the submatrix
        const int m = chainep::slot_mat(st);
        const int q = (int)chainep::slot_q(st);
        const int k = q / pg.n_ops, op = q % pg.n_ops;
        const int n = args.dims[m];
        const int n16 = (n + 15) & ~15, ncol = (n + kColRound - 1) & ~(kColRound - 1);
        // m0: first COLUMN of the result tile (the MMA's M side), n0: first ROW (N side)
        const int m0 = (t % args.mt) * kTileM, n0 = (t / args.mt) * args.bn;
        if (m0 >= n || n0 >= ncol) continue;            // tile outside this submatrix
        const int kblocks = (n16 + kBK - 1) / kBK;
        push(TileCmd{m, m0, n0, min(args.bn, ncol - n0), kblocks, (n16 - (kblocks - 1) * kBK) / 16, op,
                     k | (pg.parity_from_iters ? (((args.iters[m] + 1) & 1) << 30) : 0), s, 0, 0, 0});
        gate = true;
      }
      push(TileCmd{0, 0, 0, 0, 0, 0, -1, 0, 0, 0, 0, 0});
    }
  } else if (warp == 2) {
    // ===================== TMA producer (every CTA) =====================
    if (lane == 0) {
      int stage = 0, slot = 0;
      uint32_t phase = 0, ring_phase = 0;
      for (;;) {
        mbar_wait<kPair>(&cmd_full[slot], ring_phase);
        const TileCmd c = cmds[slot];
        mbar_arrive<kPair>(&cmd_empty[slot], 0);
        if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
        if (c.op < 0) break;
        fence_proxy_async();   // other CTAs' generic-proxy writes (ordered by the scheduler's acquire) -> TMA reads
        const ChainOp &o = pg.ops[c.op];
        const int par = chainep::cmd_par(c);
        const int m = c.mat;
        const int m0 = c.m0 + NOLSM_TILE_M * (int)rank;       // this CTA's columns of the result tile
        const int my_n = kPair ? (c.nt >> 1) : c.nt;          // this CTA's share of the tile's rows (N side)
        const int n0 = c.n0 + (kPair ? my_n * (int)rank : 0);
        const bool split = (kFeat & chainep::kFeatSplitAll) != 0 || ((kFeat & chainep::kFeatSplitAny) != 0 && o.a_lo[par] >= 0);
        // only the left operand split (the right one is exact in FP16): no lo part on the M side, and the lo
        // boxes of the N side follow its hi boxes, so that one MMA can take both (see the issuer)
        const bool half = (kFeat & chainep::kFeatSplitAny) != 0 && split && o.b_lo[par] < 0;
        const int nbox = (my_n + 63) >> 6;
        const uint32_t bytes = (uint32_t)kCtas * (uint32_t)(kATileBytes * (split && !half ? 2 : 1) +
                                                            nbox * kBoxBytes * (split ? 2 : 1));
        // M side <- right operand (K-major), N side <- left operand (MN-major)
        const CUtensorMap *ma = &args.maps[o.b[par]], *mb = &args.maps[o.a[par]];
        const CUtensorMap *mal = split && !half ? &args.maps[o.b_lo[par]] : nullptr;
        const CUtensorMap *mbl = split ? &args.maps[o.a_lo[par]] : nullptr;
        const int kb_go = max(0, c.kblocks - kClaimLead);
        for (int kb = 0; kb < c.kblocks; ++kb) {
          if (leader && kb == kb_go) mbar_arrive<false>(&claim_go);   // the scheduler may claim the next tile
          mbar_wait<kPair>(&empty_bar[stage], phase ^ 1u);
          uint8_t *st = smem + (size_t)stage * args.stage_bytes;
          if (leader) mbar_expect_tx(&full_bar[stage], bytes);
          const int k0 = kb * kBK;
          tma_load_3d<kPair>(st, ma, &full_bar[stage], k0, m0, m);
          tma_load_3d<kPair>(st + kBoxBytes, ma, &full_bar[stage], k0, m0 + 64, m);
          for (int j = 0; j < nbox; ++j)
            tma_load_3d<kPair>(st + off_b + j * kBoxBytes, mb, &full_bar[stage], n0 + 64 * j, k0, m);
          if (split) {
            if (!half) {
              tma_load_3d<kPair>(st + off_a_lo, mal, &full_bar[stage], k0, m0, m);
              tma_load_3d<kPair>(st + off_a_lo + kBoxBytes, mal, &full_bar[stage], k0, m0 + 64, m);
            }
            for (int j = 0; j < nbox; ++j)
              tma_load_3d<kPair>(st + off_b_lo + j * kBoxBytes, mbl, &full_bar[stage], n0 + 64 * j, k0, m);
          }
          if (++stage == args.stages) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA; for both CTAs of a pair) =====================
    // The whole warp walks the tile sequence (uniform control flow, operands in uniform registers); one
    // elected lane issues the MMAs, commits and arrivals.
    if (leader) {
      const bool one = elect_one();
      int stage = 0, slot = 0, acc = 0;
      uint32_t phase = 0, ring_phase = 0, acc_phase = 0;
      const uint32_t smem_base = smem_u32(smem);
      // high half of every operand descriptor: stride offset 1024 B (8-row atoms), version 1, 128-byte swizzle
      constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);
      for (;;) {
        mbar_wait<kPair>(&cmd_full[slot], ring_phase);
        const TileCmd c = cmds[slot];
        __syncwarp();
        if (one) mbar_arrive<kPair>(&cmd_empty[slot], 0);
        if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
        if (c.op < 0) break;
        const bool split = (kFeat & chainep::kFeatSplitAll) != 0 ||
                           ((kFeat & chainep::kFeatSplitAny) != 0 && pg.ops[c.op].a_lo[chainep::cmd_par(c)] >= 0);
        const bool half = (kFeat & chainep::kFeatSplitAny) != 0 && split && pg.ops[c.op].b_lo[chainep::cmd_par(c)] < 0;
        // split, one CTA, 128-row tiles: the lo boxes of the N side start exactly 128 rows behind the hi boxes, and
        // the correction accumulator 128 columns behind the main one -- ONE MMA of N = 128 + nt forms
        // [A_hi B_hi | A_hi B_lo] and reads the M-side tile once (columns nt..127 are never read back); a full
        // split adds A_lo B_hi to the correction accumulator with a second MMA
        const bool stacked = split && !kPair && args.b_bytes == 2 * kBoxBytes;
        // instruction descriptor: D=F32, A=B=F16, A K-major, B MN-major, N = nt, M = 128 per CTA
        const uint32_t idesc = (1u << 4) | (1u << 16) | ((uint32_t)(c.nt >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
        const uint32_t idesc_stacked =
            (1u << 4) | (1u << 16) | ((uint32_t)((128 + c.nt) >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
        mbar_wait<kPair>(&tempty_bar[acc], acc_phase ^ 1u);
        tc_fence_after();
        const uint32_t d_main = tmem_base + (uint32_t)(acc * 256);
        const uint32_t d_corr = d_main + 128;
        for (int kb = 0; kb < c.kblocks; ++kb) {
          mbar_wait<kPair>(&full_bar[stage], phase);
          tc_fence_after();
          // descriptor low halves: (address >> 4) | leading offset << 16; A (K-major): leading offset 16 B, +32 B
          // per K=16 step; B (MN-major): leading offset = the next 64-row chunk (8192 B), +2048 B per step
          const uint32_t sa = smem_base + (uint32_t)stage * (uint32_t)args.stage_bytes;
          const uint32_t a_lo = ((sa >> 4) & 0x3FFFu) | (1u << 16);
          const uint32_t b_lo = (((sa + off_b) >> 4) & 0x3FFFu) | ((uint32_t)(kBoxBytes >> 4) << 16);
          const int steps = kb == c.kblocks - 1 ? c.ktail : kBK / 16;
          if (one) {
            if (!split || (stacked && half)) {
              const uint32_t id = stacked ? idesc_stacked : idesc;
              tc_mma<kPair>(d_main, a_lo, b_lo, kDescHi, id, kb ? 1u : 0u);
              if (steps > 1) tc_mma<kPair>(d_main, a_lo + 2u, b_lo + 128u, kDescHi, id, 1u);
              if (steps > 2) tc_mma<kPair>(d_main, a_lo + 4u, b_lo + 256u, kDescHi, id, 1u);
              if (steps > 3) tc_mma<kPair>(d_main, a_lo + 6u, b_lo + 384u, kDescHi, id, 1u);
            } else if (stacked) {
              const uint32_t al_lo = (((sa + off_a_lo) >> 4) & 0x3FFFu) | (1u << 16);
              for (int k4 = 0; k4 < steps; ++k4) {
                tc_mma<kPair>(d_main, a_lo + 2u * k4, b_lo + 128u * k4, kDescHi, idesc_stacked, (kb | k4) ? 1u : 0u);
                tc_mma<kPair>(d_corr, al_lo + 2u * k4, b_lo + 128u * k4, kDescHi, idesc, 1u);
              }
            } else {
              const uint32_t al_lo = (((sa + off_a_lo) >> 4) & 0x3FFFu) | (1u << 16);
              const uint32_t bl_lo = (((sa + off_b_lo) >> 4) & 0x3FFFu) | ((uint32_t)(kBoxBytes >> 4) << 16);
              for (int k4 = 0; k4 < steps; ++k4) {
                const uint32_t accum = (kb | k4) ? 1u : 0u;
                tc_mma<kPair>(d_main, a_lo + 2u * k4, b_lo + 128u * k4, kDescHi, idesc, accum);
                tc_mma<kPair>(d_corr, a_lo + 2u * k4, bl_lo + 128u * k4, kDescHi, idesc, accum);
                if (!half) tc_mma<kPair>(d_corr, al_lo + 2u * k4, b_lo + 128u * k4, kDescHi, idesc, 1u);
              }
            }
            tc_commit<kPair>(&empty_bar[stage]);
          }
          __syncwarp();
          if (++stage == args.stages) { stage = 0; phase ^= 1u; }
        }
        if (one) tc_commit<kPair>(&tfull_bar[acc]);
        __syncwarp();
        if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      }
    }
  } else if (warp >= kFirstEpiWarp) {
    // ===================== epilogue compute (every CTA drains its own 128 TMEM lanes) =====================
    const int q = warp & 3;          // TMEM lane quadrant this warp may access
    const int h = (warp - kFirstEpiWarp) >> 2;   // row half of every 64-row chunk
    int slot = 0, acc = 0, tile_par = 0;
    uint32_t ring_phase = 0, acc_phase = 0;
    uint32_t uses[2] = {0u, 0u};
    for (;;) {
      mbar_wait<kPair>(&cmd_full[slot], ring_phase);
      const TileCmd c = cmds[slot];
      __syncwarp();
      if (lane == 0) mbar_arrive<kPair>(&cmd_empty[slot], 0);
      if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
      if (c.op < 0) break;
      // the peer's half of the last pair tile may lie beyond the leading dimension: nothing to load or store
      const bool rows_in = c.m0 + NOLSM_TILE_M * (int)rank < args.ld;
      chainep::EpiTile t;
      if (rows_in) chainep::epi_begin<kFeat>(args, c, c.m0 + NOLSM_TILE_M * (int)rank + q * 32 + lane, h, t);
      mbar_wait<kPair>(&tfull_bar[acc], acc_phase);
      tc_fence_after();
      const uint32_t t_main = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * 256);
      float ss = 0.f;
      auto release = [&]() {   // this warp has read its part of the accumulator stage
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive<kPair>(&tempty_bar[acc], 0);
      };
      if (rows_in) ss = chainep::epi_chunks(args, c, t, t_main, lane, q * 32 + lane, staging, ebars, uses, release);
      else release();
      if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      if (rows_in && t.o->resid) {
        for (int d = 16; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
        if (lane == 0) atomicAdd(&args.resid2[(size_t)(chainep::cmd_iter(c) % NOLSM_MAX_RESID_SLOTS) * args.count + c.mat], ss);
        // column sums of |E| (thread = column; two threads, one per row half, and ntl tiles add to a column): the
        // add returns the running total, and the largest running total of the product is its largest column sum
        const int kk = chainep::cmd_iter(c);
        // (in fixed point, 2^-20: integer sums do not depend on the order of the atomics, so that what is derived from
        // the norm is bitwise reproducible)
        if (t.colnorm && args.colsum != nullptr && kk < args.colslots) {
          unsigned int tot = 0u;
          if (t.col < t.n) {
            const unsigned int mine = (unsigned int)fminf(t.abs_sum * chainep::kColFix, 4.0e9f);
            tot = atomicAdd(&args.colsum[((size_t)kk * args.count + c.mat) * args.ld + t.col], mine) + mine;
          }
          for (int d = 16; d > 0; d >>= 1) tot = max(tot, __shfl_xor_sync(0xffffffffu, tot, d));
          if (lane == 0) atomicMax(&args.colmax[(size_t)kk * args.count + c.mat], tot);
        }
      }
      // this warp's direct stores and residual atomic are issued: join the tile's completion
      __syncwarp();
      if (lane == 0) chainep::ebar_arrive(&ebars.tile_done[tile_par]);
      tile_par ^= 1;
    }
  } else {
    // ===================== epilogue agent (one thread) =====================
    if (lane == 0) {
      const CUtensorMap *emaps = args.maps + args.n_half;
      int slot = 0;
      uint32_t ring_phase = 0, tile_seq = 0;
      uint32_t uses[2] = {0u, 0u};
      // take the next command and open its tile (both staging buffers must be free)
      auto take = [&](TileCmd &c) {
        c = cmds[slot];
        mbar_arrive<kPair>(&cmd_empty[slot], 0);
        if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
        if (c.op < 0) return;
        fence_proxy_async();   // other CTAs' writes (ordered by the scheduler's acquire) -> TMA reads of the add-in
        const int col0 = c.m0 + NOLSM_TILE_M * (int)rank;   // first column of this CTA's part of the tile
        if (col0 < args.ld) chainep::epi_agent_open(args, c, emaps, staging, ebars, col0);
      };
      TileCmd c, cn;
      mbar_wait<kPair>(&cmd_full[slot], ring_phase);
      take(c);
      while (c.op >= 0) {
        const int col0 = c.m0 + NOLSM_TILE_M * (int)rank;
        if (col0 < args.ld) chainep::epi_agent_run(args, c, emaps, staging, ebars, col0, uses);
        // Both staging buffers are free again.  If the next tile's command is already there, open that tile
        // BEFORE publishing this one: the publication (store completion, fences, atomics: ~3000 cycles) then
        // overlaps the compute warps' work on the next tile instead of delaying it.  Never wait for the next
        // command here: it may depend on this tile's publication.
        const bool have_next = mbar_test<kPair>(&cmd_full[slot], ring_phase);
        if (have_next) take(cn);
        chainep::bulk_wait0();   // this tile's TMA stores are complete
        // wait until every compute warp has issued its direct stores and residual atomic, then publish
        chainep::ebar_wait(&ebars.tile_done[tile_seq & 1u], (tile_seq >> 1) & 1u);
        ++tile_seq;
        chainep::epi_complete<kTileM, kColRound, kCtas>(args, c);
        if (!have_next) {
          mbar_wait<kPair>(&cmd_full[slot], ring_phase);
          take(cn);
        }
        c = cn;
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if constexpr (kPair) cluster_sync();   // nobody leaves while the peer may still signal our barriers or read our smem
  if (threadIdx.x == 0) atomicMax(&args.sched[3], (int32_t)((clock64() - t_start) >> 10));   // statistics only
  if (warp == 1) {
    tc_fence_after();
    if constexpr (kPair)
      asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols) : "memory");
    else
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols) : "memory");
  }
}

// The instantiations that exist: the sign iteration / plain one-shot products (0), all-split programs of the FP32 mode,
// the Eq. 15-17 chain with its column norms, the half-split residual R, the shifted B1 -> X0 product, and everything.
typedef void (*ChainKernel)(const ChainArgs);
constexpr int kNumInst = 8;
const int kInstFeat[kNumInst] = {0, chainep::kFeatSplitAll, chainep::kFeatColNorm, chainep::kFeatSplitAny,
                                 chainep::kFeatShift, chainep::kFeatRescale,
                                 chainep::kFeatSplitAll | chainep::kFeatRescale, chainep::kFeatFull};
template <bool kPair>
static ChainKernel chain_kernel_of(int feat) {
  switch (feat) {
    case 0: return k_chain<kPair, 0>;
    case chainep::kFeatSplitAll: return k_chain<kPair, chainep::kFeatSplitAll>;
    case chainep::kFeatColNorm: return k_chain<kPair, chainep::kFeatColNorm>;
    case chainep::kFeatSplitAny: return k_chain<kPair, chainep::kFeatSplitAny>;
    case chainep::kFeatShift: return k_chain<kPair, chainep::kFeatShift>;
    case chainep::kFeatRescale: return k_chain<kPair, chainep::kFeatRescale>;
    case chainep::kFeatSplitAll | chainep::kFeatRescale:
      return k_chain<kPair, chainep::kFeatSplitAll | chainep::kFeatRescale>;
    default: return k_chain<kPair, chainep::kFeatFull>;
  }
}
static ChainKernel chain_kernel(bool pair, int feat) {
  return pair ? chain_kernel_of<true>(feat) : chain_kernel_of<false>(feat);
}

// Reset of the per-launch control state: slots 0..window-1 hold submatrices 0..window-1 at product 0.
__global__ void __launch_bounds__(256)
k_chain_reset(int count, int window, unsigned long long *slot_state, int32_t *slot_done, int32_t *sched,
              int32_t *state, unsigned long long *tile_counter, float *resid2, int resid_elems, int32_t *iters,
              float *lastres, int touch_stats) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) {
    *tile_counter = 0ull;
    sched[0] = window;
    sched[1] = 0;
    sched[2] = 0;
    sched[3] = 0;
  }
  const int stride = gridDim.x * blockDim.x;
  for (int m = i; m < count; m += stride) {
    state[m] = 0x7fffffff;
    if (touch_stats) { iters[m] = 0; lastres[m] = -1.f; }
  }
  for (int s = i; s < window; s += stride) {
    slot_state[s] = chainep::slot_pack(0u, 0u, (uint32_t)s);
    slot_done[s] = 0;
  }
  for (int e = i; e < resid_elems; e += stride) resid2[e] = 0.f;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

// stored matrix: dim0 = row index (contiguous), dim1 = column index, dim2 = submatrix
// FP16 operand buffer: {64 storage rows, 64 storage columns} box with 128-byte swizzle, one map serving
// both operand roles (see the header comment)
nolsm_status encode_map(nolsm_ctx *ctx, CUtensorMap *map, void *ptr, int ld, int count, unsigned box_rows,
                        unsigned box_cols, bool swizzle, bool fp32) {
  const size_t es = fp32 ? sizeof(float) : sizeof(__half);
  cuuint64_t dims[3] = {(cuuint64_t)ld, (cuuint64_t)ld, (cuuint64_t)count};
  cuuint64_t strides[2] = {(cuuint64_t)ld * es, (cuuint64_t)ld * ld * es};
  cuuint32_t box[3] = {box_rows, box_cols, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = reinterpret_cast<EncodeTiledFn>(ctx->encode_tiled)(
      map, fp32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, ptr, dims, strides, box, estr,
      CU_TENSOR_MAP_INTERLEAVE_NONE,
      swizzle ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    ctx->err = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r);
    return NOLSM_ECUDA;
  }
  return NOLSM_OK;
}

// all pairs must be co-resident: the CTAs wait on one another through global flags
void pair_init(nolsm_ctx *ctx) {
  ctx->pair_ok = false;
  cudaError_t e = cudaSuccess;
  for (int i = 0; i < kNumInst && e == cudaSuccess; ++i)
    e = cudaFuncSetAttribute(reinterpret_cast<const void *>(chain_kernel(true, kInstFeat[i])),
                             cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit);
  if (e != cudaSuccess) { cudaGetLastError(); return; }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(ctx->sm_count & ~1));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = kSmemLimit;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  int max_clusters = 0;
  e = cudaOccupancyMaxActiveClusters(&max_clusters, k_chain<true, chainep::kFeatFull>, &cfg);
  if (e != cudaSuccess || max_clusters < 1) { cudaGetLastError(); return; }
  ctx->pair_clusters = std::min(max_clusters, ctx->sm_count / 2);
  ctx->pair_ok = true;
}

}  // namespace

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
  e = cudaSuccess;
  for (int i = 0; i < kNumInst && e == cudaSuccess; ++i)
    e = cudaFuncSetAttribute(reinterpret_cast<const void *>(chain_kernel(false, kInstFeat[i])),
                             cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit);
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
  pair_init(ctx);   // optional: the single-CTA instantiation is the fallback
  return NOLSM_OK;
}

nolsm_status umma_make_maps(nolsm_ctx *ctx, nolsm_batch *b) {
  b->maps_valid = false;
  if (!ctx->umma_ok || b->count == 0) return NOLSM_OK;
  // [0, n_half): operand maps ({64 x 64} boxes, 128-byte swizzle); [n_half, 2 n_half): epilogue maps of the same
  // buffers ({64 rows x 128 columns} boxes, 128-byte swizzle: the staging planes of chain_epilogue.cuh)
  std::vector<CUtensorMap> maps(2 * b->n_half + b->n_unit);
  for (int i = 0; i < b->n_half; ++i) {
    nolsm_status s = encode_map(ctx, &maps[i], b->h[i], b->ld, b->count, 64, 64, true, false);
    if (s == NOLSM_OK)
      s = encode_map(ctx, &maps[b->n_half + i], b->h[i], b->ld, b->count, chainep::kChunkRows, 128, true, false);
    if (s != NOLSM_OK) return s;
  }
  // FP32 units: {32 rows x 128 columns} boxes for results that leave through the staging buffers
  for (int i = 0; i < b->n_unit; ++i) {
    nolsm_status s = encode_map(ctx, &maps[2 * b->n_half + i], b->u[i], b->ld, b->count, 32, 128, true, true);
    if (s != NOLSM_OK) return s;
  }
  if (!b->d_maps) {
    if (cudaMalloc(&b->d_maps, sizeof(CUtensorMap) * (2 * NOLSM_MAX_HALF + NOLSM_MAX_UNIT)) != cudaSuccess) {
      cudaGetLastError();
      ctx->err = "cudaMalloc of the tensor maps failed";
      return NOLSM_ENOMEM;
    }
  }
  NOLSM_CUDA(ctx, cudaMemcpy(b->d_maps, maps.data(), sizeof(CUtensorMap) * maps.size(), cudaMemcpyHostToDevice));
  b->maps_valid = true;
  return NOLSM_OK;
}

// The instantiation that runs a program: the one whose feature set is exactly what the program needs if it exists
// (kInstFeat), else the full kernel
static int program_features(const ChainProgram &prog) {
  using namespace chainep;
  int need = prog.use_alpha_tab ? kFeatAlphaTab : 0;
  int n_full_split = 0, n_plain = 0;
  for (int i = 0; i < prog.n_ops; ++i) {
    const ChainOp &o = prog.ops[i];
    if (o.cin32 >= 0 || o.cout32 >= 0) need |= kFeatFp32;
    if (o.colnorm == 1) need |= kFeatColNorm;
    if (o.colnorm == 2) need |= kFeatRescale;
    if (o.diag != 0.f || o.use_div == 2) need |= kFeatShift;
    const bool s0 = o.a_lo[0] >= 0 && o.b_lo[0] >= 0, s1 = o.a_lo[1] >= 0 && o.b_lo[1] >= 0;
    const bool p0 = o.a_lo[0] < 0 && o.b_lo[0] < 0, p1 = o.a_lo[1] < 0 && o.b_lo[1] < 0;
    if (s0 && s1) ++n_full_split;
    else if (p0 && p1) ++n_plain;
  }
  if (n_full_split == prog.n_ops) need |= kFeatSplitAll;
  else if (n_plain != prog.n_ops) need |= kFeatSplitAny;
  for (int i = 0; i < kNumInst; ++i)
    if (kInstFeat[i] == need) return need;
  return kFeatFull;
}

// Runs `prog` over every submatrix of the batch.  touch_stats: reset and fill iters / lastres.
cudaError_t launch_chain(nolsm_ctx *ctx, const nolsm_batch *b, const ChainProgram &prog, const float *alpha_div,
                         bool touch_stats, cudaStream_t st) {
  if (b->count == 0) return cudaSuccess;
  if (!ctx->umma_ok || !b->maps_valid) return cudaErrorNotSupported;
  const int forced = ctx->cfg.flags & (NOLSM_FLAG_PAIR | NOLSM_FLAG_SINGLE);
  const bool pair = ctx->pair_ok && ((forced & NOLSM_FLAG_PAIR) || (forced == 0 && b->prefer_pair));
  ChainArgs a;
  memset(&a, 0, sizeof(a));
  a.prog = prog;
  bool split = false, full_split = false;   // full: both operands split (lo tiles on both sides of a stage)
  for (int i = 0; i < prog.n_ops; ++i) {
    split |= prog.ops[i].a_lo[0] >= 0 || prog.ops[i].a_lo[1] >= 0;
    full_split |= prog.ops[i].b_lo[0] >= 0 || prog.ops[i].b_lo[1] >= 0;
  }
  const int col_round = pair ? 32 : 16;
  const int ncol_max = (b->max_n + col_round - 1) / col_round * col_round;
  const int tile_m = pair ? 2 * NOLSM_TILE_M : NOLSM_TILE_M;
  a.bn = std::min(split ? 128 : 256, ncol_max);
  a.b_bytes = (((pair ? a.bn >> 1 : a.bn) + 63) / 64) * kBoxBytes;
  a.stage_bytes = full_split ? 2 * (kATileBytes + a.b_bytes) : kATileBytes + a.b_bytes * (split ? 2 : 1);
  a.stages = std::min(kMaxStages, (kSmemLimit - 1024 - chainep::kStagingBytes) / a.stage_bytes);
  a.mt = (b->max_n + tile_m - 1) / tile_m;
  a.ntl = (ncol_max + a.bn - 1) / a.bn;
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
  a.window = std::max(1, std::min(prog.group, b->count));
  a.prog.group = a.window;
  a.slot_state = b->d_slot_state;
  a.slot_done = b->d_slot_done;
  a.sched = b->d_sched;
  a.state = b->d_state;
  a.iters = b->d_iters;
  a.alpha_tab = prog.use_alpha_tab ? b->d_alpha : nullptr;
  a.alpha_rt = prog.use_alpha_tab ? nullptr : b->d_alpha;   // (the two scalings exclude one another)
  a.tile_counter = b->d_tile_counter;
  a.resid2 = b->d_resid2;
  a.colsum = nullptr;
  a.colmax = nullptr;
  a.colslots = 0;
  const int strips = colpart_strips(b->ld);   // d_colpart: strips * count * ld floats (norm-bound scratch, free here)
  for (int i = 0; i < prog.n_ops; ++i)
    if (prog.ops[i].colnorm) {   // strips - 1 iteration slots of column sums, the last strip: maxima
      a.colsum = reinterpret_cast<unsigned int *>(b->d_colpart);
      a.colslots = strips - 1;
      a.colmax = reinterpret_cast<unsigned int *>(b->d_colpart + (size_t)(strips - 1) * b->count * b->ld);
    }
  a.lastres = b->d_lastres;
  const int slots = std::min(prog.max_iter, NOLSM_MAX_RESID_SLOTS);
  k_chain_reset<<<64, 256, 0, st>>>(b->count, a.window, a.slot_state, a.slot_done, a.sched, a.state, a.tile_counter,
                                    a.resid2, slots * b->count, a.iters, a.lastres, touch_stats ? 1 : 0);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (a.colsum != nullptr) {
    e = cudaMemsetAsync(a.colsum, 0, sizeof(float) * (size_t)strips * b->count * b->ld, st);
    if (e != cudaSuccess) return e;
  }
  const size_t smem_bytes = (size_t)(a.stages * a.stage_bytes + chainep::kStagingBytes + 1024);
  const int feat = program_features(prog);
  if (!pair) {
    void *params[] = {&a};
    return cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(chain_kernel(false, feat)), dim3(ctx->sm_count),
                                       dim3(kThreads), params, smem_bytes, st);
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(2 * ctx->pair_clusters));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem_bytes;
  cfg.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeCooperative;
  at[1].val.cooperative = 1;
  cfg.attrs = at;
  cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, chain_kernel(true, feat), a);
}
