// nolsm_build_neighbours_static: a0 (neighbour lists) for callers that cannot allocate device memory
// (tight serving loops, harnesses that forbid cudaMalloc, code that must not touch the allocator).  Same kernels and
// same result as nolsm_build_neighbours; the one piece of scratch that entry point takes from cudaMalloc -- the
// per-molecule neighbour counts between the counting pass and the prefix sum -- lives in a file-scope device array
// here, of a fixed maximum size.
//
// The array exists once per device that loads the library (NOLSM_STATIC_MAX_MOL * 4 bytes = 1 MiB, held until the
// process exits) and is SHARED by every call on that device: calls that overlap on the GPU (two streams, two host
// threads) race on it.  Serialise them.  Nothing in it has to start at zero: the counting pass writes counts[j] for
// every j < n_mol before the prefix sum reads them, so the contents a previous call left behind are never read.
#include <mutex>

#include "common.cuh"

// In host code this name is only a handle for cudaGetSymbolAddress, never a device address.
static __device__ __align__(256) int32_t g_neighbour_counts[NOLSM_STATIC_MAX_MOL];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_mutex;
int32_t *g_counts_addr[kMaxDevices];   // device address of g_neighbour_counts, per device ordinal

// Set-up, once per device, with that device current: the device address of the scratch array.
cudaError_t counts_address(int32_t **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mutex);
  if (g_counts_addr[dev] == nullptr) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_neighbour_counts);
    if (e != cudaSuccess) return e;
    g_counts_addr[dev] = static_cast<int32_t *>(p);
  }
  *out = g_counts_addr[dev];
  return cudaSuccess;
}

nolsm_status fail(nolsm_ctx *ctx, nolsm_status rc, const std::string &msg) {
  if (ctx) ctx->err = msg;
  return rc;
}

}  // namespace

extern "C" nolsm_status nolsm_static_setup(void) {
  int32_t *p = nullptr;
  if (counts_address(&p) != cudaSuccess) { cudaGetLastError(); return NOLSM_ECUDA; }
  return NOLSM_OK;
}

extern "C" nolsm_status nolsm_build_neighbours_static(nolsm_ctx *ctx, int32_t n_mol, const int32_t *pos_q,
                                                      const int32_t *box_q, int32_t rc_q, int32_t *row_ptr,
                                                      int32_t *col_idx, int64_t cap, int64_t *nnzb_out,
                                                      void *stream) {
  if (n_mol < 0 || !row_ptr || !box_q || (n_mol > 0 && !pos_q) || rc_q < 0 || cap < 0)
    return fail(ctx, NOLSM_EINVAL, "nolsm_build_neighbours_static: bad argument");
  if (n_mol > NOLSM_STATIC_MAX_MOL)
    return fail(ctx, NOLSM_EINVAL, "nolsm_build_neighbours_static: n_mol = " + std::to_string(n_mol) +
                                       " exceeds NOLSM_STATIC_MAX_MOL = " + std::to_string(NOLSM_STATIC_MAX_MOL) +
                                       " (the static scratch array); use nolsm_build_neighbours");
  for (int a = 0; a < 3; ++a)
    if (box_q[a] <= 0 || (box_q[a] & 1)) return fail(ctx, NOLSM_EINVAL, "box lengths must be positive and even");
  cudaStream_t st = (cudaStream_t)stream;
  int32_t *counts = nullptr;
  cudaError_t e = counts_address(&counts);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return fail(ctx, NOLSM_ECUDA, std::string("cudaGetSymbolAddress of the static scratch: ") + cudaGetErrorString(e));
  }
  e = launch_neighbour_count(n_mol, pos_q, box_q, rc_q, counts, st);
  if (e == cudaSuccess) e = launch_exclusive_scan(counts, row_ptr, n_mol, st);
  int32_t total = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&total, row_ptr + n_mol, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (ctx) ctx->launches += 2;
  if (e != cudaSuccess) {
    cudaGetLastError();
    return fail(ctx, NOLSM_ECUDA, std::string("neighbour count: ") + cudaGetErrorString(e));
  }
  if (nnzb_out) *nnzb_out = total;
  if ((int64_t)total > cap || (total > 0 && !col_idx)) return fail(ctx, NOLSM_ENOMEM, "col_idx capacity too small");
  e = launch_neighbour_fill(n_mol, pos_q, box_q, rc_q, row_ptr, col_idx, st);
  if (ctx) ctx->launches += 1;
  if (e != cudaSuccess) {
    cudaGetLastError();
    return fail(ctx, NOLSM_ECUDA, std::string("neighbour fill: ") + cudaGetErrorString(e));
  }
  return NOLSM_OK;
}
