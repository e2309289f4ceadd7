// whp_static.cu — the one entry point of the library that allocates nothing: a7 (D7, argmin with
// ties to the lowest index) for callers that cannot reach cudaMalloc (code under CUDA graph
// capture, tight serving loops, harnesses that forbid it). Every other call of include/whp.h
// works on a whp_ctx, whose creation allocates; this one needs no context.
//
// The block-then-grid reduction of whp_argmin.cu needs scratch: one (value, index) pair per
// block and the ticket that elects the last block. Here that scratch is a file-scope
// __device__ array of a fixed size — every GPU that loads libwhp.so holds its
// WHP_ARGMIN_STATIC_SCRATCH_BYTES until the process exits — so the size of a call is bounded:
// a block reduces one fixed chunk of kChunk values, the array has room for kMaxParts blocks,
// n <= WHP_ARGMIN_STATIC_MAX_N = kMaxParts * kChunk.
//
// In HOST code the array's name is a host-side stand-in, not a device address. The device
// address comes from cudaGetSymbolAddress, asked once per device with that device current
// (device_scratch below), and is what the kernel and the ticket's memset are given.
//
// All calls share the array and it keeps the last call's contents: the ticket is cleared on the
// stream before every launch (a call that was torn down half-way cannot poison the next one),
// the pairs are always written before they are read. Two calls that OVERLAP on the GPU (two
// streams, or two host threads on two streams) race on it: serialise them.
#include <cuda_runtime.h>

#include <climits>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/whp.h"

namespace {

constexpr int kThreads = 256;
constexpr int kPerThread = 16;
constexpr int kChunk = kThreads * kPerThread;  // values per block
constexpr int kMaxParts = 4096;                // blocks the scratch has room for
constexpr int kMaxDevices = 64;

static_assert((int64_t)kMaxParts * kChunk == WHP_ARGMIN_STATIC_MAX_N, "header and kernel disagree");

struct pair_t { double v; int64_t i; };

struct scratch_t {
  pair_t part[kMaxParts];
  unsigned ticket;  // blocks that have stored their pair; zero when a launch starts
  unsigned pad[63];
};
static_assert(sizeof(scratch_t) == WHP_ARGMIN_STATIC_SCRATCH_BYTES, "header and kernel disagree");

static __device__ __align__(256) unsigned char g_scratch[sizeof(scratch_t)];

__device__ __forceinline__ bool less_than(double v1, int64_t i1, double v2, int64_t i2) {
  return v1 < v2 || (v1 == v2 && i1 < i2);  // D7: ties go to the lowest index
}

__device__ __forceinline__ void warp_reduce(double& v, int64_t& i) {
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) {
    const double v2 = __shfl_xor_sync(0xffffffffu, v, off);
    const int64_t i2 = __shfl_xor_sync(0xffffffffu, i, off);
    if (less_than(v2, i2, v, i)) { v = v2; i = i2; }
  }
}

// every lane of warp 0 returns the block's minimum; sh holds one pair per warp
__device__ __forceinline__ void block_reduce(double& v, int64_t& i, pair_t* sh) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  warp_reduce(v, i);
  if (lane == 0) { sh[warp].v = v; sh[warp].i = i; }
  __syncthreads();
  if (warp == 0) {
    const pair_t p = sh[lane < kThreads / 32 ? lane : 0];  // a repeat of sh[0] changes nothing
    v = p.v; i = p.i;
    warp_reduce(v, i);
  }
}

// grid = ceil(n / kChunk) <= kMaxParts blocks; block b reduces x[b*kChunk, (b+1)*kChunk) ∩ [0, n)
__global__ void __launch_bounds__(kThreads)
whp_argmin_static_kernel(const double* __restrict__ x, int64_t n, scratch_t* __restrict__ s,
                         int64_t* __restrict__ d_idx, double* __restrict__ d_val) {
  __shared__ pair_t sh[kThreads / 32];
  __shared__ bool last;
  const int64_t lo = (int64_t)blockIdx.x * kChunk;  // < n by the grid size
  double v = __ldg(x + lo);
  int64_t i = lo;
#pragma unroll 4
  for (int t = 0; t < kPerThread; ++t) {
    const int64_t k = lo + (int64_t)t * kThreads + threadIdx.x;
    if (k < n) {
      const double xv = __ldg(x + k);
      if (less_than(xv, k, v, i)) { v = xv; i = k; }
    }
  }
  block_reduce(v, i, sh);
  if (threadIdx.x == 0) {
    s->part[blockIdx.x].v = v;
    s->part[blockIdx.x].i = i;
    __threadfence();
    last = (atomicAdd(&s->ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  v = __ldcg(&s->part[0].v);
  i = __ldcg(&s->part[0].i);
  for (int k = threadIdx.x; k < (int)gridDim.x; k += kThreads) {
    const double pv = __ldcg(&s->part[k].v);
    const int64_t pi = __ldcg(&s->part[k].i);
    if (less_than(pv, pi, v, i)) { v = pv; i = pi; }
  }
  __syncthreads();  // sh is reused
  block_reduce(v, i, sh);
  if (threadIdx.x == 0) {
    *d_idx = i;
    if (d_val) *d_val = v;
  }
}

thread_local char t_err[256] = "";

whp_status fail(whp_status st, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess)
    std::snprintf(t_err, sizeof t_err, "%s: %s", what, cudaGetErrorString(e));
  else
    std::snprintf(t_err, sizeof t_err, "%s", what);
  return st;
}

// the device address of g_scratch on the CURRENT device, asked once per device
std::mutex g_mu;
scratch_t* g_dev_scratch[kMaxDevices] = {};

whp_status device_scratch(scratch_t** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(WHP_ERR_CUDA, "cudaGetDevice", e);
  if (dev < 0 || dev >= kMaxDevices)
    return fail(WHP_ERR_OUT_OF_RANGE, "whp_argmin_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_dev_scratch[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_scratch);
    if (e != cudaSuccess) return fail(WHP_ERR_CUDA, "cudaGetSymbolAddress(g_scratch)", e);
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255u))
      return fail(WHP_ERR_CUDA, "whp_argmin_static: scratch address is null or misaligned");
    g_dev_scratch[dev] = static_cast<scratch_t*>(p);
  }
  *out = g_dev_scratch[dev];
  return WHP_OK;
}

}  // namespace

extern "C" {

whp_status whp_argmin_static_setup(void) {
  scratch_t* s = nullptr;
  const whp_status st = device_scratch(&s);
  if (st == WHP_OK) t_err[0] = 0;
  return st;
}

whp_status whp_argmin_static(const double* d_obj, int64_t n, int64_t* d_idx, double* d_val,
                             void* cuda_stream) {
  if (!d_obj || !d_idx) return fail(WHP_ERR_INVALID_ARG, "whp_argmin_static: null d_obj or d_idx");
  if (n < 1) return fail(WHP_ERR_INVALID_ARG, "whp_argmin_static: n must be >= 1");
  if (n > WHP_ARGMIN_STATIC_MAX_N) {
    std::snprintf(t_err, sizeof t_err,
                  "whp_argmin_static: n = %lld exceeds WHP_ARGMIN_STATIC_MAX_N = %lld (the static "
                  "scratch holds %d block results of %d values); use whp_argmin",
                  (long long)n, (long long)WHP_ARGMIN_STATIC_MAX_N, kMaxParts, kChunk);
    return WHP_ERR_OUT_OF_RANGE;
  }
  scratch_t* s = nullptr;
  const whp_status st = device_scratch(&s);
  if (st != WHP_OK) return st;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  cudaError_t e = cudaMemsetAsync(&s->ticket, 0, sizeof(unsigned), stream);
  if (e != cudaSuccess) return fail(WHP_ERR_CUDA, "cudaMemsetAsync(ticket)", e);
  const unsigned blocks = (unsigned)((n + kChunk - 1) / kChunk);
  whp_argmin_static_kernel<<<blocks, kThreads, 0, stream>>>(d_obj, n, s, d_idx, d_val);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(WHP_ERR_CUDA, "whp_argmin_static_kernel launch", e);
  t_err[0] = 0;
  return WHP_OK;
}

const char* whp_static_last_error(void) { return t_err; }

}  // extern "C"
