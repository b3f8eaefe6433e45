// Pair-CTA variant of the matrix-iteration engine (see chain_umma.cu for the scheduling, the
// dependency protocol and the epilogues, which are identical): two CTAs of a cluster (one TPC)
// compute ONE 256 x N tile with tcgen05.mma.cta_group::2.  Each CTA stages its own 128 rows of the A
// operand and only HALF of the B operand's columns, so the operand bytes an SM must take in per
// 64-deep K block drop from 48 KB (128 x 256 tile, cta_group::1) to 32 KB.  That delivery rate, not the
// tensor pipe, bounds the single-CTA kernel (profiles/r1_k_chain_sign_w32768.md).
//
// Protocol differences to chain_umma.cu:
//   * the scheduler runs in the leader CTA (cluster rank 0) only and writes every tile command into
//     both CTAs' rings (st.shared::cluster + remote mbarrier arrive), so the two CTAs can never
//     disagree on the tile sequence;
//   * `full` (operands landed) and `tmem empty` barriers live in the leader: both CTAs' TMA loads
//     signal the leader's `full` barrier (cp.async.bulk.tensor ... cta_group::2), the peer's epilogue
//     warps arrive remotely on `tmem empty`;
//   * the leader's single MMA thread issues for both CTAs and releases smem stages / publishes the
//     accumulator in both CTAs with tcgen05.commit ... multicast::cluster.
#include "common.cuh"
#include "chain_epilogue.cuh"

namespace pair {

using chainep::TileCmd;
typedef chainep::ChainArgs PairArgs;

constexpr int kThreads = 352;
constexpr int kEpiWarps = 8;
constexpr int kBK = 64;
constexpr int kMaxStages = 8;
constexpr int kTmemCols = 512;
constexpr int kBoxBytes = 64 * 128;
constexpr int kATileBytes = 2 * kBoxBytes;     // this CTA's 128 rows x 64 K
constexpr int kRing = 2;
constexpr int kSmemLimit = 232448 - 2048;
constexpr int32_t kDone = 0x7fffffff;
constexpr int kTileM = 256;                    // rows of a pair tile

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
// arrive on a barrier given by its shared::cluster address (own or peer CTA), release at cluster scope
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// wait with acquire at cluster scope (the arrivals may come from the peer CTA)
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
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
}
// TMA load into THIS CTA's shared memory that signals the barrier at shared::cluster address `bar`
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, uint32_t bar, int c0, int c1,
                                            int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.cta_group::2.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, "
      "{%3, %4, %5}], [%2];" ::"r"(smem_u32(dst)),
      "l"(reinterpret_cast<uint64_t>(map)), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// arrives on the barrier at the same offset in BOTH CTAs once all prior MMAs of this thread are done
__device__ __forceinline__ void tc_commit_both(uint64_t *bar) {
  asm volatile(
      "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
          smem_u32(bar)),
      "h"((uint16_t)3)
      : "memory");
}
// descriptors as 32-bit halves (constant high half, low half = base + k * step): few integer instructions
// per MMA for the issuing lane (see chain_umma.cu)
__device__ __forceinline__ void tc_mma_lh(uint32_t tmem_d, uint32_t a_lo, uint32_t b_lo, uint32_t desc_hi,
                                          uint32_t idesc, uint32_t accumulate) {
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
}
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
__device__ __forceinline__ int32_t ld_acquire(const int32_t *p) {
  int32_t v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
#ifdef NOLSM_TRACE
__device__ long long g_ptrace[4][4096][2];
__device__ long long g_pwait[4096][4];
#define PTRACE(role, ti, j) do { if (blockIdx.x == 0 && (ti) < 4096) g_ptrace[role][ti][j] = clock64(); } while (0)
#define PTRACEV(role, ti, j, v) do { if (blockIdx.x == 0 && (ti) < 4096) g_ptrace[role][ti][j] = (v); } while (0)
#else
#define PTRACE(role, ti, j)
#define PTRACEV(role, ti, j, v)
#endif

__global__ void __launch_bounds__(kThreads, 1) k_chain_pair(const PairArgs args) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ uint64_t full_bar[kMaxStages], empty_bar[kMaxStages], tfull_bar[2], tempty_bar[2];
  __shared__ uint64_t cmd_full[kRing], cmd_empty[kRing];
  __shared__ __align__(16) TileCmd cmds[kRing];
  __shared__ uint32_t tmem_base_s;

  const ChainProgram &pg = args.prog;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_rank();
  const bool leader = rank == 0;
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  // stage layout: [A hi 16K][B hi b_bytes][A lo 16K][B lo b_bytes]
  const int off_b = kATileBytes, off_a_lo = kATileBytes + args.b_bytes, off_b_lo = 2 * kATileBytes + args.b_bytes;

  if (threadIdx.x == 0) {
    for (int s = 0; s < args.stages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(&tfull_bar[a], 1); mbar_init(&tempty_bar[a], 2 * kEpiWarps); }
    // command ring: filled by the leader's scheduler in both CTAs; freed (leader's barrier) by the
    // leader's MMA issuer + both TMA producers + both CTAs' epilogue warps
    for (int r = 0; r < kRing; ++r) { mbar_init(&cmd_full[r], 1); mbar_init(&cmd_empty[r], 3 + 2 * kEpiWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                 "r"(kTmemCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync();          // barriers of both CTAs initialised before any remote arrive / multicast commit
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;

  if (warp == 0) {
    // ===================== scheduler (leader CTA only) =====================
    if (leader && lane == 0) {
      int slot = 0;
      uint32_t ring_phase = 0;
      const int T = args.mt * args.ntl;
      const int limit = pg.fixed_iter > 0 ? min(pg.fixed_iter, pg.max_iter) : pg.max_iter;
      const int n_groups = (args.count + pg.group - 1) / pg.group;
      const int n_clusters = gridDim.x >> 1, cluster_id = blockIdx.x >> 1;
      auto push = [&](const TileCmd &cmd) {
        mbar_wait(&cmd_empty[slot], ring_phase ^ 1u);
        cmds[slot] = cmd;
        const uint32_t remote = mapa(smem_u32(&cmds[slot]), 1);
        asm volatile("st.shared::cluster.v4.s32 [%0], {%1, %2, %3, %4};" ::"r"(remote), "r"(cmd.mat), "r"(cmd.m0),
                     "r"(cmd.n0), "r"(cmd.nt)
                     : "memory");
        asm volatile("st.shared::cluster.v4.s32 [%0], {%1, %2, %3, %4};" ::"r"(remote + 16), "r"(cmd.kblocks),
                     "r"(cmd.ktail), "r"(cmd.op), "r"(cmd.iter)
                     : "memory");
        mbar_arrive_cluster(mapa(smem_u32(&cmd_full[slot]), 0));
        mbar_arrive_cluster(mapa(smem_u32(&cmd_full[slot]), 1));
        if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
      };
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
        const int n16 = (n + 15) & ~15, n32 = (n + 31) & ~31;
        const int m0 = (t % args.mt) * kTileM, n0 = (t / args.mt) * args.bn;
        if (m0 >= n || n0 >= n32) continue;          // tile outside this submatrix
        const int need = k * pg.n_ops + op;          // ops of this submatrix that must be complete
        if (need > 0) {
          int32_t r = ld_acquire(&args.ready[m]);
          while (r < need) { __nanosleep(64); r = ld_acquire(&args.ready[m]); }
          if (r == kDone) continue;                  // submatrix finished at an earlier iteration
        }
        const int kblocks = (n16 + kBK - 1) / kBK;
        {
          push(TileCmd{m, m0, n0, min(args.bn, n32 - n0), kblocks, (n16 - (kblocks - 1) * kBK) / 16, op,
                          k | (pg.parity_from_iters ? (((args.iters[m] + 1) & 1) << 30) : 0)});
        }
      }
      push(TileCmd{0, 0, 0, 0, 0, 0, -1, 0});
    }
  } else if (warp == 2) {
    // ===================== TMA producer (both CTAs) =====================
    if (lane == 0) {
#ifdef NOLSM_TRACE
      int tti = 0;
#endif
      int stage = 0, slot = 0;
      uint32_t phase = 0, ring_phase = 0;
      for (;;) {
        mbar_wait(&cmd_full[slot], ring_phase);
        const TileCmd c = cmds[slot];
        mbar_arrive_cluster(mapa(smem_u32(&cmd_empty[slot]), 0));
        if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
        if (c.op < 0) break;
        PTRACE(2, tti, 0);
        fence_proxy_async();   // other CTAs' generic-proxy writes (ordered by the scheduler's acquire) -> TMA reads
        const ChainOp &o = pg.ops[c.op];
        const int par = chainep::cmd_par(c);
        const int m = c.mat;
        const int m0 = c.m0 + 128 * (int)rank;               // this CTA's rows of the pair tile
        const int half_n = c.nt >> 1;
        const int n0 = c.n0 + half_n * (int)rank;            // this CTA's half of the B columns
        const bool split = o.a_lo[par] >= 0;
        const int nbox = (half_n + 63) >> 6;
        const uint32_t bytes = 2u * (uint32_t)(kATileBytes + nbox * kBoxBytes) * (split ? 2u : 1u);  // both CTAs
        const CUtensorMap *ma = &args.maps[o.a[par]], *mb = &args.maps[o.b[par]];
        const CUtensorMap *mal = split ? &args.maps[o.a_lo[par]] : nullptr;
        const CUtensorMap *mbl = split ? &args.maps[o.b_lo[par]] : nullptr;
        for (int kb = 0; kb < c.kblocks; ++kb) {
          mbar_wait(&empty_bar[stage], phase ^ 1u);
          uint8_t *st = smem + (size_t)stage * args.stage_bytes;
          if (leader) mbar_expect_tx(&full_bar[stage], bytes);
          const uint32_t fb = mapa(smem_u32(&full_bar[stage]), 0);
          const int k0 = kb * kBK;
          tma_load_3d(st, ma, fb, m0, k0, m);
          tma_load_3d(st + kBoxBytes, ma, fb, m0 + 64, k0, m);
          for (int j = 0; j < nbox; ++j) tma_load_3d(st + off_b + j * kBoxBytes, mb, fb, k0, n0 + 64 * j, m);
          if (split) {
            tma_load_3d(st + off_a_lo, mal, fb, m0, k0, m);
            tma_load_3d(st + off_a_lo + kBoxBytes, mal, fb, m0 + 64, k0, m);
            for (int j = 0; j < nbox; ++j)
              tma_load_3d(st + off_b_lo + j * kBoxBytes, mbl, fb, k0, n0 + 64 * j, m);
          }
          if (++stage == args.stages) { stage = 0; phase ^= 1u; }
        }
        PTRACE(2, tti, 1);
#ifdef NOLSM_TRACE
        ++tti;
#endif
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only, for both CTAs) =====================
    if (leader) {   // whole warp, uniform control flow; one elected lane issues (see chain_umma.cu)
      const bool one = elect_one();
      const uint32_t smem_base = smem_u32(smem);
      constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);
#ifdef NOLSM_TRACE
      int mti = 0;
#endif
      int stage = 0, slot = 0, acc = 0;
      uint32_t phase = 0, ring_phase = 0, acc_phase = 0;
      for (;;) {
        mbar_wait(&cmd_full[slot], ring_phase);
        const TileCmd c = cmds[slot];
        __syncwarp();
        if (one) mbar_arrive_cluster(mapa(smem_u32(&cmd_empty[slot]), 0));
        if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
        if (c.op < 0) break;
        const bool split = pg.ops[c.op].a_lo[chainep::cmd_par(c)] >= 0;
        // instruction descriptor: D=F32, A=B=F16, A M-major, B K-major, N = nt, M = 256 (128 per CTA)
        const uint32_t idesc = (1u << 4) | (1u << 15) | ((uint32_t)(c.nt >> 3) << 17) | ((256u >> 4) << 24);
        PTRACE(0, mti, 0);
        mbar_wait(&tempty_bar[acc], acc_phase ^ 1u);
        tc_fence_after();
        PTRACE(0, mti, 1);
#ifdef NOLSM_TRACE
        ++mti;
#endif
        const uint32_t d_main = tmem_base + (uint32_t)(acc * 256);
        const uint32_t d_corr = d_main + 128;
#ifdef NOLSM_TRACE
        long long wsum = 0, t_first = 0, t_begin = clock64();
#endif
        for (int kb = 0; kb < c.kblocks; ++kb) {
#ifdef NOLSM_TRACE
          long long w0 = clock64();
#endif
          mbar_wait(&full_bar[stage], phase);
#ifdef NOLSM_TRACE
          wsum += clock64() - w0;
          if (kb == 0) t_first = clock64() - w0;
#endif
          tc_fence_after();
          const uint32_t sa = smem_base + (uint32_t)stage * (uint32_t)args.stage_bytes;
          const uint32_t a_lo = ((sa >> 4) & 0x3FFFu) | ((uint32_t)(kBoxBytes >> 4) << 16);
          const uint32_t b_lo = (((sa + off_b) >> 4) & 0x3FFFu) | (1u << 16);
          const int steps = kb == c.kblocks - 1 ? c.ktail : kBK / 16;
          if (one) {
            if (!split) {
              if (steps > 0) tc_mma_lh(d_main, a_lo, b_lo, kDescHi, idesc, kb ? 1u : 0u);
              if (steps > 1) tc_mma_lh(d_main, a_lo + 128u, b_lo + 2u, kDescHi, idesc, 1u);
              if (steps > 2) tc_mma_lh(d_main, a_lo + 256u, b_lo + 4u, kDescHi, idesc, 1u);
              if (steps > 3) tc_mma_lh(d_main, a_lo + 384u, b_lo + 6u, kDescHi, idesc, 1u);
            } else {
              const uint32_t al_lo = (((sa + off_a_lo) >> 4) & 0x3FFFu) | ((uint32_t)(kBoxBytes >> 4) << 16);
              const uint32_t bl_lo = (((sa + off_b_lo) >> 4) & 0x3FFFu) | (1u << 16);
              for (int k4 = 0; k4 < steps; ++k4) {
                const uint32_t accum = (kb | k4) ? 1u : 0u;
                tc_mma_lh(d_main, a_lo + 128u * k4, b_lo + 2u * k4, kDescHi, idesc, accum);
                tc_mma_lh(d_corr, a_lo + 128u * k4, bl_lo + 2u * k4, kDescHi, idesc, accum);
                tc_mma_lh(d_corr, al_lo + 128u * k4, b_lo + 2u * k4, kDescHi, idesc, 1u);
              }
            }
            tc_commit_both(&empty_bar[stage]);
          }
          __syncwarp();
          if (++stage == args.stages) { stage = 0; phase ^= 1u; }
        }
        if (one) tc_commit_both(&tfull_bar[acc]);
        __syncwarp();
#ifdef NOLSM_TRACE
        if (blockIdx.x == 0 && mti - 1 < 4096) { g_pwait[mti - 1][0] = wsum; g_pwait[mti - 1][1] = t_first; g_pwait[mti - 1][2] = clock64() - t_begin; }
#endif
        if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      }
    }
  } else {
    // ===================== epilogue (both CTAs: each drains its own 128 TMEM lanes) =====================
    const int q = warp & 3;
    const int chunk_first = (warp - 3) >> 2;
#ifdef NOLSM_TRACE
    int eti = 0;
#endif
    int slot = 0, acc = 0, tile_seq = 0;
    uint32_t ring_phase = 0, acc_phase = 0;
    for (;;) {
      mbar_wait(&cmd_full[slot], ring_phase);
      const TileCmd c = cmds[slot];
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(mapa(smem_u32(&cmd_empty[slot]), 0));
      if (++slot == kRing) { slot = 0; ring_phase ^= 1u; }
      if (c.op < 0) break;
      // the peer's half of the last pair tile may lie beyond the leading dimension: nothing to load or store
      const bool rows_in = c.m0 + 128 * (int)rank < args.ld;
      chainep::EpiTile t;
      chainep::epi_begin(args, c, c.m0 + 128 * (int)rank + q * 32, rows_in, lane, chunk_first, t);
      if (warp == 3 && lane == 0) { PTRACE(1, eti, 0); }
      mbar_wait(&tfull_bar[acc], acc_phase);
      tc_fence_after();
      if (warp == 3 && lane == 0) { PTRACE(1, eti, 1); PTRACEV(3, eti, 0, ((long long)c.mat << 40) | ((long long)c.iter << 32) | ((long long)c.op << 24) | ((long long)(c.m0 / 256) << 8) | (long long)(c.n0 / 64)); }
      const uint32_t t_main = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * 256);
      float ss = chainep::epi_chunks(args, c, t, t_main, lane);
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(mapa(smem_u32(&tempty_bar[acc]), 0));
      if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      if (t.o->resid) {
        for (int d = 16; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
        if (lane == 0) atomicAdd(&args.resid2[(size_t)(chainep::cmd_iter(c) % NOLSM_MAX_RESID_SLOTS) * args.count + c.mat], ss);
      }
      // all epilogue warps of this CTA have issued their stores: one thread publishes the CTA's half
      asm volatile("bar.sync 1, %0;" ::"n"(kEpiWarps * 32) : "memory");
      if (warp - 3 == (tile_seq & (kEpiWarps - 1)) && lane == 0) chainep::epi_complete<kTileM, 32, 2>(args, c);
      ++tile_seq;
      if (warp == 3 && lane == 0) { PTRACE(3, eti, 1); }
#ifdef NOLSM_TRACE
      ++eti;
#endif
    }
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync();            // nobody leaves while the peer may still signal our barriers or read our smem
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols) : "memory");
  }
}

}  // namespace pair

#ifdef NOLSM_TRACE
extern "C" void nolsm_debug_ptrace(long long *host_out) {
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(host_out, pair::g_ptrace, sizeof(pair::g_ptrace));
}
extern "C" void nolsm_debug_pwait(long long *host_out) { cudaMemcpyFromSymbol(host_out, pair::g_pwait, sizeof(pair::g_pwait)); }
#endif

nolsm_status pair_init(nolsm_ctx *ctx) {
  ctx->pair_ok = false;
  cudaError_t e = cudaFuncSetAttribute(pair::k_chain_pair, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       pair::kSmemLimit);
  if (e != cudaSuccess) { cudaGetLastError(); return NOLSM_ECUDA; }
  // all pairs must be co-resident: the CTAs wait on one another through global flags
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(ctx->sm_count & ~1));
  cfg.blockDim = dim3(pair::kThreads);
  cfg.dynamicSmemBytes = pair::kSmemLimit;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  int max_clusters = 0;
  e = cudaOccupancyMaxActiveClusters(&max_clusters, pair::k_chain_pair, &cfg);
  if (e != cudaSuccess || max_clusters < 1) { cudaGetLastError(); return NOLSM_ECUDA; }
  ctx->pair_clusters = std::min(max_clusters, ctx->sm_count / 2);
  ctx->pair_ok = true;
  return NOLSM_OK;
}

// Same contract as the single-CTA launch in chain_umma.cu; the control state has been reset by the caller.
cudaError_t launch_chain_pair(nolsm_ctx *ctx, const nolsm_batch *b, const ChainProgram &prog, const float *alpha_div,
                              cudaStream_t st) {
  using namespace pair;
  PairArgs a;
  memset(&a, 0, sizeof(a));
  a.prog = prog;
  bool split = false;
  for (int i = 0; i < prog.n_ops; ++i) split |= prog.ops[i].a_lo[0] >= 0 || prog.ops[i].a_lo[1] >= 0;
  const int n32max = (b->max_n + 31) & ~31;
  a.bn = std::min(split ? 128 : 256, n32max);
  a.b_bytes = (((a.bn >> 1) + 63) / 64) * kBoxBytes;
  a.stage_bytes = (kATileBytes + a.b_bytes) * (split ? 2 : 1);
  a.stages = std::min(kMaxStages, (kSmemLimit - 1024) / a.stage_bytes);
  a.mt = (b->max_n + kTileM - 1) / kTileM;
  a.ntl = (n32max + a.bn - 1) / a.bn;
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
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(2 * ctx->pair_clusters));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = (size_t)(a.stages * a.stage_bytes + 1024);
  cfg.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeCooperative;
  at[1].val.cooperative = 1;
  cfg.attrs = at;
  cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, k_chain_pair, a);
}
