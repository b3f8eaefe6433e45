// Batched n x n x n products on the 5th-generation tensor cores (tcgen05 + TMEM + TMA), sm_100a only.
//
// Every GEMM of the matrix iterations (Eq. 9-10, Eq. 15-17) goes
// through this kernel: FP16 operands, FP32 accumulation in TMEM, FP32 master iterate updated in the
// epilogue ("FP16 with FP32-based accumulation"; master iterates: DESIGN.md reading 12).
//
// Layout facts this kernel relies on:
//   * all matrices are column-major, so the A operand (M x K) is M-major ("MN-major") and the B operand
//     (K x N) is K-major in shared memory; one TMA tensor map per buffer serves both roles with two
//     boxes: {64 rows, 64 cols} (A role, two boxes per 128-row tile) and {64 rows, bn cols} (B role).
//   * 128-byte swizzle everywhere: smem rows are 64 FP16 = 128 B; 8-row atoms of 1024 B.
//   * accumulator: 128 TMEM lanes = tile rows, one 32-bit column per tile column; the epilogue thread
//     that owns lane r therefore writes element (r, c) for successive c, and a warp-wide store covers
//     32 consecutive rows of one column = contiguous in column-major memory.
//
// Warp roles (192 threads): warp 0 = TMA producer, warp 1 = MMA issuer (+ TMEM allocation),
// warps 2..5 = epilogue (TMEM lane quadrant = warp_id % 4).  Persistent over a static tile list.
#include "common.cuh"

namespace {

constexpr int kThreads = 192;
constexpr int kBK = 64;              // K elements per pipeline stage (= one 128-byte swizzle row)
constexpr int kMaxStages = 8;
constexpr int kTmemCols = 512;
constexpr int kSmemBytes = 200 * 1024;   // > half of the SM's shared memory: one CTA per SM, so the
                                         // 512-column TMEM allocation can never contend
constexpr int kAChunkBytes = 64 * 128;   // one {64 x 64} FP16 box
constexpr int kATileBytes = 2 * kAChunkBytes;

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
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(
                   smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void tc_mma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                           uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}\n" ::"r"(tmem_d),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&v)[32]) {
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
__device__ __forceinline__ void tc_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor (tcgen05): start address, leading / stride byte offsets (all >> 4),
// descriptor version 1, 128-byte swizzle.
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;   // version
  d |= (uint64_t)2 << 61;   // SWIZZLE_128B
  return d;
}

struct UmmaArgs {
  GemmParams p;
  int32_t kind;        // 1 = FP16 operands, 2 = split (hi/lo) operands
  int32_t bn;          // B box width (columns loaded per stage)
  int32_t stages;
  int32_t stage_bytes; // bytes of one stage (A + B, hi [+ lo])
  uint32_t lbo_a, sbo_a, sbo_b;   // descriptor offsets (bytes)
};

__global__ void __launch_bounds__(kThreads, 1)
k_gemm_umma(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
            const __grid_constant__ CUtensorMap map_a_lo, const __grid_constant__ CUtensorMap map_b_lo,
            const UmmaArgs args) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ uint64_t full_bar[kMaxStages], empty_bar[kMaxStages], tfull_bar[2], tempty_bar[2];
  __shared__ uint32_t tmem_base_s;

  const GemmParams &p = args.p;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const bool split = args.kind == 2;
  const int b_tile_bytes = args.bn * 128;
  // stage layout: [A hi 16K][B hi bn*128][A lo 16K][B lo bn*128]
  const int off_b = kATileBytes, off_a_lo = kATileBytes + b_tile_bytes, off_b_lo = 2 * kATileBytes + b_tile_bytes;

  if (threadIdx.x == 0) {
    for (int s = 0; s < args.stages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(&tfull_bar[a], 1); mbar_init(&tempty_bar[a], 4); }
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
    // ===================== TMA producer =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
        const TileDesc td = p.tiles[t];
        if (p.state && p.iter > p.state[td.mat]) continue;
        const int n = p.dims[td.mat];
        const int kblocks = (n + kBK - 1) / kBK;
        const uint32_t bytes = (uint32_t)(kATileBytes + b_tile_bytes) * (split ? 2u : 1u);
        for (int kb = 0; kb < kblocks; ++kb) {
          mbar_wait(&empty_bar[stage], phase ^ 1u);
          uint8_t *st = smem + (size_t)stage * args.stage_bytes;
          mbar_expect_tx(&full_bar[stage], bytes);
          const int k0 = kb * kBK;
          tma_load_3d(st, &map_a, &full_bar[stage], td.m0, k0, td.mat);
          tma_load_3d(st + kAChunkBytes, &map_a, &full_bar[stage], td.m0 + 64, k0, td.mat);
          tma_load_3d(st + off_b, &map_b, &full_bar[stage], k0, td.n0, td.mat);
          if (split) {
            tma_load_3d(st + off_a_lo, &map_a_lo, &full_bar[stage], td.m0, k0, td.mat);
            tma_load_3d(st + off_a_lo + kAChunkBytes, &map_a_lo, &full_bar[stage], td.m0 + 64, k0, td.mat);
            tma_load_3d(st + off_b_lo, &map_b_lo, &full_bar[stage], k0, td.n0, td.mat);
          }
          if (++stage == args.stages) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      int acc = 0;
      uint32_t acc_phase = 0;
      for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
        const TileDesc td = p.tiles[t];
        if (p.state && p.iter > p.state[td.mat]) continue;
        const int n = p.dims[td.mat];
        const int kblocks = (n + kBK - 1) / kBK;
        // instruction descriptor: D=F32, A=B=F16, A M-major, B K-major, N = td.nt, M = 128
        const uint32_t idesc = (1u << 4) | (1u << 15) | ((uint32_t)(td.nt >> 3) << 17) | ((128u >> 4) << 24);
        mbar_wait(&tempty_bar[acc], acc_phase ^ 1u);
        tc_fence_after();
        const uint32_t d_main = tmem_base + (uint32_t)(acc * 256);
        const uint32_t d_corr = d_main + 128;
        for (int kb = 0; kb < kblocks; ++kb) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + (size_t)stage * args.stage_bytes);
#pragma unroll
          for (int k4 = 0; k4 < kBK / 16; ++k4) {
            // A (M-major): 16 K-rows of 128 B per MMA -> +2048 B; B (K-major): 16 K elements -> +32 B
            const uint64_t ad = make_smem_desc(sa + k4 * 2048, args.lbo_a, args.sbo_a);
            const uint64_t bd = make_smem_desc(sa + off_b + k4 * 32, 16, args.sbo_b);
            const uint32_t accum = (kb | k4) ? 1u : 0u;
            tc_mma_f16(d_main, ad, bd, idesc, accum);
            if (split) {
              const uint64_t adl = make_smem_desc(sa + off_a_lo + k4 * 2048, args.lbo_a, args.sbo_a);
              const uint64_t bdl = make_smem_desc(sa + off_b_lo + k4 * 32, 16, args.sbo_b);
              tc_mma_f16(d_corr, ad, bdl, idesc, accum);
              tc_mma_f16(d_corr, adl, bd, idesc, 1u);
            }
          }
          tc_commit(&empty_bar[stage]);
          if (++stage == args.stages) { stage = 0; phase ^= 1u; }
        }
        tc_commit(&tfull_bar[acc]);
        if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      }
    }
  } else {
    // ===================== epilogue =====================
    const int q = warp & 3;          // TMEM lane quadrant this warp may access
    int acc = 0;
    uint32_t acc_phase = 0;
    for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
      const TileDesc td = p.tiles[t];
      if (p.state && p.iter > p.state[td.mat]) continue;
      const int n = p.dims[td.mat];
      const int r = td.m0 + q * 32 + lane;
      const int64_t base = (int64_t)td.mat * p.slab + r;
      const float alpha = p.alpha_div ? p.alpha / p.alpha_div[td.mat] : p.alpha;
      mbar_wait(&tfull_bar[acc], acc_phase);
      tc_fence_after();
      const uint32_t t_main = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * 256);
      float ss = 0.f;
      for (int c0 = 0; c0 < td.nt; c0 += 32) {
        uint32_t v[32];
        tc_ld32(t_main + c0, v);
        tc_ld_wait();
        if (split) {
          uint32_t w[32];
          tc_ld32(t_main + 128 + c0, w);
          tc_ld_wait();
#pragma unroll
          for (int j = 0; j < 32; ++j)
            v[j] = __float_as_uint(fmaf(__uint_as_float(w[j]), 1.f / 2048.f, __uint_as_float(v[j])));
        }
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const int c = td.n0 + c0 + j;
          const int64_t off = base + (int64_t)c * p.ld;
          const float a = __uint_as_float(v[j]);
          float o;
          if (p.mode == EPI_IDENT) {
            o = ((r == c) ? 1.f : 0.f) - a;
            if (r < n && c < n) ss = fmaf(o, o, ss);
          } else {
            o = alpha * a;
            if (p.beta != 0.f) o = fmaf(p.beta, p.cin32[off], o);
          }
          if (p.cout32) p.cout32[off] = o;
          if (p.cout16) {
            const __half hi = __float2half_rn(o);
            p.cout16[off] = hi;
            if (p.cout16_lo) p.cout16_lo[off] = __float2half_rn((o - __half2float(hi)) * 2048.f);
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tempty_bar[acc]);
      if (p.mode == EPI_IDENT && p.resid2) {
        for (int d = 16; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
        if (lane == 0) atomicAdd(&p.resid2[td.mat], ss);
      }
      if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols) : "memory");
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

nolsm_status encode_map(nolsm_ctx *ctx, CUtensorMap *map, __half *ptr, int ld, int count, int box_rows,
                        int box_cols) {
  // stored matrix: dim0 = row index (contiguous), dim1 = column index, dim2 = submatrix
  cuuint64_t dims[3] = {(cuuint64_t)ld, (cuuint64_t)ld, (cuuint64_t)count};
  cuuint64_t strides[2] = {(cuuint64_t)ld * sizeof(__half), (cuuint64_t)ld * ld * sizeof(__half)};
  cuuint32_t box[3] = {(cuuint32_t)box_rows, (cuuint32_t)box_cols, 1};
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

// Debug knobs for bring-up on hardware (descriptor offsets); 0 = built-in value.
static uint32_t g_lbo_a = 0, g_sbo_a = 0, g_sbo_b = 0;
extern "C" void nolsm_debug_set_desc(uint32_t lbo_a, uint32_t sbo_a, uint32_t sbo_b) {
  g_lbo_a = lbo_a; g_sbo_a = sbo_a; g_sbo_b = sbo_b;
}

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
  e = cudaFuncSetAttribute(k_gemm_umma, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  if (e != cudaSuccess) {
    ctx->err = std::string("cudaFuncSetAttribute(k_gemm_umma): ") + cudaGetErrorString(e);
    cudaGetLastError();
    return NOLSM_ECUDA;
  }
  ctx->umma_ok = true;
  return NOLSM_OK;
}

nolsm_status umma_make_maps(nolsm_ctx *ctx, nolsm_batch *b) {
  b->maps_valid = false;
  if (!ctx->umma_ok || b->count == 0) return NOLSM_OK;
  for (int i = 0; i < 6; ++i) {
    nolsm_status s = encode_map(ctx, &b->map_a[i], b->h[i], b->ld, b->count, 64, 64);
    if (s != NOLSM_OK) return s;
    s = encode_map(ctx, &b->map_b[i], b->h[i], b->ld, b->count, 64, b->bn);
    if (s != NOLSM_OK) return s;
  }
  b->maps_valid = true;
  return NOLSM_OK;
}

cudaError_t launch_gemm_umma(nolsm_ctx *ctx, const nolsm_batch *b, int kind, int a_buf, int b_buf,
                             int a_lo_buf, int b_lo_buf, const GemmParams &p, cudaStream_t st) {
  if (p.n_tiles == 0) return cudaSuccess;
  if (!ctx->umma_ok || !b->maps_valid) return cudaErrorNotSupported;
  UmmaArgs a;
  a.p = p;
  a.kind = kind;
  a.bn = b->bn;
  a.stage_bytes = (kATileBytes + b->bn * 128) * (kind == 2 ? 2 : 1);
  int stages = (kSmemBytes - 1024) / a.stage_bytes;
  a.stages = stages > kMaxStages ? kMaxStages : stages;
  a.lbo_a = g_lbo_a ? g_lbo_a : (uint32_t)kAChunkBytes;  // between the two 64-row chunks of the A tile
  a.sbo_a = g_sbo_a ? g_sbo_a : 1024u;                   // between 8-row K atoms
  a.sbo_b = g_sbo_b ? g_sbo_b : 1024u;                   // between 8-row N atoms
  const int grid = p.n_tiles < ctx->sm_count ? p.n_tiles : ctx->sm_count;
  const int al = kind == 2 ? a_lo_buf : a_buf, bl = kind == 2 ? b_lo_buf : b_buf;
  k_gemm_umma<<<grid, kThreads, kSmemBytes, st>>>(b->map_a[a_buf], b->map_b[b_buf], b->map_a[al],
                                                  b->map_b[bl], a);
  return cudaGetLastError();
}
