// Epilogue of the matrix-iteration engine, shared by the single-CTA kernel (chain_umma.cu) and the
// pair-CTA kernel (chain_pair.cu): one epilogue warp drains its 32 TMEM lanes (= 32 rows) of the tile
// in 32-column chunks, applies the fused epilogue of the op
//     EPI_IDENT :  E = I - A B,  ||E||_F^2 over the true n x n part (stop rule, reading 9)
//     EPI_AXPBY :  C = beta * C32 + alpha * A B   (FP32 master update, reading 12)
// and writes the FP32 result and the FP16 operand copies (hi [, lo * 2^11]) with coalesced stores: the
// lanes of a warp hold consecutive rows, so every store instruction writes one contiguous 128-byte
// (FP32) or 64-byte (FP16) segment of a column.  Measured store rate of an SM into L2 with this
// pattern: ~29 B/clk (FP32), ~20 B/clk (FP16) -- the floor of the epilogue (profiles/r1_k_chain_sign_w32768.md).
//
// Completion protocol (per submatrix and op): after the stores of a tile the epilogue warps of the
// CTA meet at a named barrier and ONE elected thread makes them visible (__threadfence) and adds 1 to
// tiles_done[m]; the arrival that completes the op evaluates the stop rule and publishes ready[m].
// (One fence + one atomic round trip cost ~3000 cycles; paid by one warp per tile, not by all eight.)
#pragma once
#include "common.cuh"

// store flavours (experiments: -DNOLSM_ST=1 streaming .cs, 2 write-through .wt, 3 .cg)
#if NOLSM_ST == 1
#define ST32(p, v) __stcs((p), (v))
#define ST16(p, v) __stcs(reinterpret_cast<unsigned short *>(p), __half_as_ushort(v))
#elif NOLSM_ST == 2
#define ST32(p, v) __stwt((p), (v))
#define ST16(p, v) __stwt(reinterpret_cast<unsigned short *>(p), __half_as_ushort(v))
#elif NOLSM_ST == 3
#define ST32(p, v) __stcg((p), (v))
#define ST16(p, v) __stcg(reinterpret_cast<unsigned short *>(p), __half_as_ushort(v))
#else
#define ST32(p, v) (*(p) = (v))
#define ST16(p, v) (*(p) = (v))
#endif

namespace chainep {

constexpr int32_t kDone = 0x7fffffff;

struct TileCmd {              // scheduler -> TMA producer(s), MMA issuer and epilogue warps
  int32_t mat, m0, n0, nt;    // submatrix, first row / column of the tile, tile columns
  int32_t kblocks, ktail;     // K blocks of 64; K=16 steps in the last one (1..4)
  int32_t op, iter;           // op < 0: no more tiles
};

// TileCmd::iter carries the iteration in its low bits and, in bit 30, a flip of the operand-table parity
// (ChainProgram::parity_from_iters).
__device__ __forceinline__ int cmd_iter(const TileCmd &c) { return c.iter & 0x3fffffff; }
__device__ __forceinline__ int cmd_par(const TileCmd &c) { return (c.iter ^ (c.iter >> 30)) & 1; }

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
  int32_t *ready, *tiles_done, *state, *iters, *group_active;
  unsigned long long *tile_counter;   // next tile index to claim (dynamic scheduling)
  float *resid2, *lastres;
  // scaled Newton-Schulz start (nolsm_config.gap_hint): alpha_tab[m * kAlphaSteps + k] = alpha_k of submatrix m
  // for iteration k < kAlphaSteps (1 afterwards); null = the plain iteration
  const float *alpha_tab;
};
constexpr int kAlphaSteps = 8;

__device__ __forceinline__ uint32_t s32(const void *p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
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
__device__ __forceinline__ void ld_tmem_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void st_release_gpu(int32_t *p, int32_t v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
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
  const int need = cmd_iter(c) * pg.n_ops + c.op;
  const int limit = pg.fixed_iter > 0 ? min(pg.fixed_iter, pg.max_iter) : pg.max_iter;
  __threadfence();      // the CTA's stores (ordered before us by the barrier) become visible GPU-wide
  const int32_t old = atomicAdd(&args.tiles_done[c.mat], 1);
  if (old + 1 != (need + 1) * tiles_m * kArrivals) return;
  __threadfence();
  const int k = cmd_iter(c);
  if (o.resid) {
    const float r2 = *reinterpret_cast<volatile float *>(
        &args.resid2[(size_t)(k % NOLSM_MAX_RESID_SLOTS) * args.count + c.mat]);
    const float res = sqrtf(fmaxf(r2, 0.f) / (float)n);
    args.lastres[c.mat] = res;
    bool stop = pg.fixed_iter > 0 ? (k + 1 >= pg.fixed_iter) : ((res < pg.tol) || !(res == res));
    // a scaled step (alpha_k > 1) measures ||I - alpha^2 X^2||, not the residual of the stop rule
    if (args.alpha_tab != nullptr && k < kAlphaSteps && pg.fixed_iter <= 0 && res == res &&
        args.alpha_tab[c.mat * kAlphaSteps + k] > 1.f)
      stop = false;
    if (k + 1 >= pg.max_iter) stop = true;
    args.iters[c.mat] = (stop && pg.stop_early) ? k : k + 1;   // iterations carried out in full
    if (stop) *reinterpret_cast<volatile int32_t *>(&args.state[c.mat]) = k;
  }
  const int32_t stv = *reinterpret_cast<volatile int32_t *>(&args.state[c.mat]);
  // stop_early: the residual product is op 0; the schedulers waiting for ops 1.. of this iteration see
  // kDone and skip their tiles
  const bool early = pg.stop_early && o.resid && stv == k;
  if (early || (c.op == pg.n_ops - 1 && (stv == k || k + 1 >= limit))) {
    st_release_gpu(&args.ready[c.mat], kDone);
    __threadfence();
    atomicSub(&args.group_active[c.mat / pg.group], 1);
  } else {
    st_release_gpu(&args.ready[c.mat], need + 1);
  }
}

// Cached per-tile epilogue parameters and the prefetch of the first FP32-master chunk; call before
// waiting for the accumulator.
struct EpiTile {
  const ChainOp *o;
  int par, n, r, nchunks, chunk_first;
  bool split, ident, has_cin, rows_in;
  float alpha, beta;
  float *p32;                 // FP32 output, element (r, first chunk column) or null
  const float *cinp;          // FP32 master input, same position, or null
  const __half *cinh;         // FP16 add-in instead (ChainOp::cin16), or null
  __half *p16, *p16l;         // FP16 outputs (hi, lo), same position, or null
  float cpre[32];
};

__device__ __forceinline__ void epi_begin(const ChainArgs &args, const TileCmd &c, int row0, bool rows_in, int lane,
                                          int chunk_first, EpiTile &t) {
  const ChainOp &o = args.prog.ops[c.op];
  t.o = &o;
  t.par = cmd_par(c);
  t.n = args.dims[c.mat];
  t.r = row0 + lane;
  t.rows_in = rows_in;
  t.nchunks = (c.nt + 31) >> 5;
  t.chunk_first = chunk_first;
  t.split = o.a_lo[t.par] >= 0;
  t.ident = o.mode == EPI_IDENT;
  const bool cin_half = o.cin16[t.par] >= 0;
  t.has_cin = !t.ident && (o.cin32 >= 0 || cin_half) && o.beta != 0.f && rows_in;
  t.alpha = o.use_div ? o.alpha / args.alpha_div[c.mat] : o.alpha;
  t.beta = o.beta;
  if (args.alpha_tab != nullptr && cmd_iter(c) < kAlphaSteps) {
    // X_{k+1} = 1/2 a X (3I - a^2 X^2):  E = I - a^2 X X,  X' = a X + (1/2 a) X E
    const float a = args.alpha_tab[c.mat * kAlphaSteps + cmd_iter(c)];
    if (t.ident) t.alpha *= a * a; else { t.alpha *= a; t.beta *= a; }
  }
  const int64_t off = (int64_t)c.mat * args.slab + t.r + (int64_t)(c.n0 + 32 * chunk_first) * args.ld;
  t.p32 = (o.cout32 >= 0 && rows_in) ? args.ubuf[o.cout32] + off : nullptr;
  t.cinp = (t.has_cin && !cin_half) ? args.ubuf[o.cin32] + off : nullptr;
  t.cinh = (t.has_cin && cin_half) ? args.hbuf[o.cin16[t.par]] + off : nullptr;
  t.p16 = (o.out16[t.par] >= 0 && rows_in) ? args.hbuf[o.out16[t.par]] + off : nullptr;
  t.p16l = (o.out16_lo[t.par] >= 0 && rows_in) ? args.hbuf[o.out16_lo[t.par]] + off : nullptr;
#if defined(NOLSM_NOEPI) || defined(NOLSM_NOCIN)   // timing experiments only (results are wrong)
  t.has_cin = false;
#endif
#ifdef NOLSM_NOSTORE
  t.p32 = nullptr; t.p16 = nullptr; t.p16l = nullptr;
#endif
#ifdef NOLSM_SCRATCHSTORE   // all stores of a CTA land in one small L2-resident region (same request count, no DRAM traffic)
  {
    const int64_t o2 = (int64_t)(blockIdx.x & 15) * args.slab + t.r % 128 + (int64_t)(32 * chunk_first) * args.ld;
    if (t.p32) t.p32 = args.ubuf[o.cout32] + o2;
    if (t.p16) t.p16 = args.hbuf[o.out16[t.par]] + o2;
    if (t.p16l) t.p16l = args.hbuf[o.out16_lo[t.par]] + o2;
  }
#endif
  if (t.has_cin && chunk_first < t.nchunks) {
    if (t.cinh) {
      const __half *ph = t.cinh;
#pragma unroll
      for (int j = 0; j < 32; ++j) { t.cpre[j] = __half2float(__ldcg(ph)); ph += args.ld; }
    } else {
      const float *pc = t.cinp;
#pragma unroll
      for (int j = 0; j < 32; ++j) { t.cpre[j] = __ldcg(pc); pc += args.ld; }
    }
  }
}

// Drains this warp's chunks of the accumulator at TMEM address t_main (lane quadrant and accumulator
// stage already applied); returns the warp's partial residual sum (lane-local; reduce before use).
__device__ __forceinline__ float epi_chunks(const ChainArgs &args, const TileCmd &c, EpiTile &t, uint32_t t_main,
                                            int lane, long long *tr = nullptr) {
#define EPI_TR(j) do { if (tr && lane == 0 && ci == t.chunk_first) tr[j] = clock64(); } while (0)
  float ss = 0.f;
  if (!t.rows_in) return ss;
#ifdef NOLSM_NOEPI   // timing experiment only: main loop without any epilogue work (results are wrong)
  return ss;
#endif
  const ChainOp &o = *t.o;
  const int64_t chunk_stride = (int64_t)32 * args.ld;
  for (int ci = t.chunk_first; ci < t.nchunks; ci += 2) {
    const int c0 = ci * 32;
    const int cnt = min(32, c.nt - c0);   // 16 or 32 valid columns
    uint32_t v[32];
    ld_tmem32(t_main + c0, v);
    if (t.split) {
      uint32_t w[32];
      ld_tmem32(t_main + 128 + c0, w);
      ld_tmem_wait();
#pragma unroll
      for (int j = 0; j < 32; ++j)
        v[j] = __float_as_uint(fmaf(__uint_as_float(w[j]), 1.f / 2048.f, __uint_as_float(v[j])));
    } else {
      ld_tmem_wait();
    }
    EPI_TR(2);
    if (t.has_cin) {
#pragma unroll
      for (int j = 0; j < 32; ++j)
        v[j] = __float_as_uint(fmaf(t.beta, t.cpre[j], t.alpha * __uint_as_float(v[j])));
      if (ci + 2 < t.nchunks) {
        if (t.cinh) {
          t.cinh += 2 * chunk_stride;
          const __half *ph = t.cinh;
#pragma unroll
          for (int j = 0; j < 32; ++j) { t.cpre[j] = __half2float(__ldcg(ph)); ph += args.ld; }
        } else {
          t.cinp += 2 * chunk_stride;
          const float *pc = t.cinp;
#pragma unroll
          for (int j = 0; j < 32; ++j) { t.cpre[j] = __ldcg(pc); pc += args.ld; }
        }
      }
    } else if (t.ident) {
      // valid columns of this chunk inside the true n x n part (residual of the stop rule)
      const int nvalid = (t.r < t.n) ? min(cnt, t.n - (c.n0 + c0)) : 0;
      const int dj = t.r - (c.n0 + c0);     // chunk column that holds the diagonal element of row r
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        const float e = fmaf(-t.alpha, __uint_as_float(v[j]), (j == dj) ? 1.f : 0.f);
        if (j < nvalid) ss = fmaf(e, e, ss);
        v[j] = __float_as_uint(e);
      }
    } else {
#pragma unroll
      for (int j = 0; j < 32; ++j) v[j] = __float_as_uint(t.alpha * __uint_as_float(v[j]));
    }
    EPI_TR(3);
    if (t.p32) {   // FP32 result: one 128-byte segment per column and warp
      float *q = t.p32;
#pragma unroll
      for (int j = 0; j < 16; ++j) { ST32(q, __uint_as_float(v[j])); q += args.ld; }
      if (cnt == 32) {
#pragma unroll
        for (int j = 16; j < 32; ++j) { ST32(q, __uint_as_float(v[j])); q += args.ld; }
      }
      t.p32 += 2 * chunk_stride;
    }
    EPI_TR(4);
    if (t.p16) {   // FP16 operand copies: one 64-byte segment per column and warp
      __half *q = t.p16, *ql = t.p16l;
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        if (j == 16 && cnt < 32) break;
        const float val = __uint_as_float(v[j]);
        const __half hi = __float2half_rn(val);
        ST16(q, hi); q += args.ld;
        if (ql) { *ql = __float2half_rn((val - __half2float(hi)) * 2048.f); ql += args.ld; }
      }
      t.p16 += 2 * chunk_stride;
      if (t.p16l) t.p16l += 2 * chunk_stride;
    }
    EPI_TR(6);
  }
#undef EPI_TR
  return ss;
}

}  // namespace chainep
