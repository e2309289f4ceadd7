// whp_argmin.cu — a7 (D7): block-then-grid argmin with a deterministic tie rule (lowest
// index), the device-side swap application of the D8 trajectory, and the permutation checker.
#include "whp_walk.cuh"

namespace {

struct am_pair { double v; int64_t i; };

__device__ __forceinline__ bool am_less(double v1, int64_t i1, double v2, int64_t i2) {
  return v1 < v2 || (v1 == v2 && i1 < i2);
}

__device__ __forceinline__ void am_warp_reduce(double& v, int64_t& i) {
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) {
    const double v2 = __shfl_xor_sync(WHP_FULL, v, off);
    const int64_t i2 = __shfl_xor_sync(WHP_FULL, i, off);
    if (am_less(v2, i2, v, i)) { v = v2; i = i2; }
  }
}

constexpr int kAmThreads = 256;

__device__ __forceinline__ void am_block_reduce(double& v, int64_t& i, am_pair* sh) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  am_warp_reduce(v, i);
  if (lane == 0) { sh[warp].v = v; sh[warp].i = i; }
  __syncthreads();
  if (warp == 0) {
    const bool has = lane < kAmThreads / 32;
    v = has ? sh[lane].v : 0.0;
    i = has ? sh[lane].i : INT64_MAX;
    if (!has) v = sh[0].v;  // neutral: never beats sh[0] (same value, larger index)
    am_warp_reduce(v, i);
  }
}

// parts: [gridDim.x] pairs followed by one unsigned ticket counter (zero between launches)
__global__ void __launch_bounds__(kAmThreads)
whp_argmin_kernel(const double* __restrict__ x, int64_t n, am_pair* parts, unsigned* ticket,
                  int64_t* __restrict__ d_idx, double* __restrict__ d_val) {
  __shared__ am_pair sh[kAmThreads / 32];
  __shared__ bool last;
  // every thread starts from element 0 (always valid) so no sentinel value is needed
  double v = __ldg(x);
  int64_t i = 0;
  for (int64_t k = (int64_t)blockIdx.x * kAmThreads + threadIdx.x; k < n;
       k += (int64_t)gridDim.x * kAmThreads) {
    const double xv = __ldg(x + k);
    if (am_less(xv, k, v, i)) { v = xv; i = k; }
  }
  am_block_reduce(v, i, sh);
  if (threadIdx.x == 0) {
    parts[blockIdx.x].v = v; parts[blockIdx.x].i = i;
    __threadfence();
    last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  v = __ldcg(&parts[0].v); i = __ldcg(&parts[0].i);
  for (int k = threadIdx.x; k < (int)gridDim.x; k += kAmThreads) {
    const double pv = __ldcg(&parts[k].v);
    const int64_t pi = __ldcg(&parts[k].i);
    if (am_less(pv, pi, v, i)) { v = pv; i = pi; }
  }
  __syncthreads();
  am_block_reduce(v, i, sh);
  if (threadIdx.x == 0) {
    *d_idx = i;
    if (d_val) *d_val = v;
    *ticket = 0;
  }
}

__global__ void whp_apply_swap_kernel(int32_t* base_perm, int32_t win_start, int32_t W,
                                      const int64_t* __restrict__ d_idx) {
  const int64_t n = *d_idx;
  if (n < 0 || n >= (int64_t)W * (W - 1) / 2) return;  // not a neighbour: leave the plan untouched
  int64_t i = 0, row = W - 1, rem = n;
  while (rem >= row && row > 0) { rem -= row; --row; ++i; }
  const int64_t j = i + 1 + rem;
  const int32_t a = base_perm[win_start + i];
  base_perm[win_start + i] = base_perm[win_start + j];
  base_perm[win_start + j] = a;
}

// one block per row; bitmap of seen order ids in dynamic shared memory
__global__ void whp_validate_kernel(const int32_t* __restrict__ perms, int64_t n_cand,
                                    int32_t n_orders, unsigned long long* n_bad) {
  extern __shared__ uint32_t seen[];
  __shared__ int bad;
  const int words = (n_orders + 31) >> 5;
  for (int64_t row = blockIdx.x; row < n_cand; row += gridDim.x) {
    for (int w = threadIdx.x; w < words; w += blockDim.x) seen[w] = 0;
    if (threadIdx.x == 0) bad = 0;
    __syncthreads();
    for (int p = threadIdx.x; p < n_orders; p += blockDim.x) {
      const int32_t o = perms[row * n_orders + p];
      if (o < 0 || o >= n_orders) { bad = 1; continue; }
      const uint32_t old = atomicOr(&seen[o >> 5], 1u << (o & 31));
      if (old & (1u << (o & 31))) bad = 1;
    }
    __syncthreads();
    if (threadIdx.x == 0 && bad) atomicAdd(n_bad, 1ull);
    __syncthreads();
  }
}

// Measurement helper (bench.py's L2 figure): `reps` read-only sweeps of an L2-resident buffer
// with 16-byte loads that bypass L1 (ld.global.cg); the xor keeps the loads alive.
__global__ void __launch_bounds__(256)
whp_l2_probe_kernel(const uint4* __restrict__ buf, int64_t n16, int32_t reps, uint32_t* __restrict__ sink) {
  uint32_t acc = 0;
  for (int32_t r = 0; r < reps; ++r)
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16;
         i += (int64_t)gridDim.x * blockDim.x) {
      const uint4 v = __ldcg(buf + i);
      acc ^= v.x ^ v.y ^ v.z ^ v.w;
    }
  if (acc == 0x9e3779b9u) *sink = acc;  // practically never: the buffer is zero-filled
}

}  // namespace

cudaError_t whp_launch_l2_probe(whp_ctx* c, int64_t bytes, int32_t reps, float* ms) {
  uint4* buf = nullptr;
  uint32_t* sink = nullptr;
  cudaError_t e = cudaMalloc(&buf, (size_t)bytes);
  if (e == cudaSuccess) e = cudaMalloc(&sink, 4);
  if (e == cudaSuccess) e = cudaMemset(buf, 0, (size_t)bytes);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (e == cudaSuccess) e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  if (e == cudaSuccess) {
    const unsigned blocks = (unsigned)c->num_sms * 8;
    whp_l2_probe_kernel<<<blocks, 256>>>(buf, bytes / 16, 2, sink);  // warm the L2
    cudaEventRecord(e0);
    whp_l2_probe_kernel<<<blocks, 256>>>(buf, bytes / 16, reps, sink);
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
    c->launches += 2;
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(buf); cudaFree(sink);
  return e;
}

cudaError_t whp_launch_argmin(whp_ctx* c, const double* d_obj, int64_t n, int64_t* d_idx,
                              double* d_val, cudaStream_t st) {
  int64_t blocks = (n + kAmThreads * 4 - 1) / (kAmThreads * 4);
  if (blocks > c->argmin_cap) blocks = c->argmin_cap;
  if (blocks < 1) blocks = 1;
  am_pair* parts = (am_pair*)c->d_argmin_part;
  unsigned* ticket = (unsigned*)(parts + c->argmin_cap);
  whp_argmin_kernel<<<(unsigned)blocks, kAmThreads, 0, st>>>(d_obj, n, parts, ticket, d_idx,
                                                             d_val);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t whp_launch_apply_swap(whp_ctx* c, int32_t* d_base_perm, int32_t win_start,
                                  int32_t win_len, const int64_t* d_idx, cudaStream_t st) {
  whp_apply_swap_kernel<<<1, 1, 0, st>>>(d_base_perm, win_start, win_len, d_idx);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t whp_launch_validate(whp_ctx* c, const int32_t* d_perms, int64_t n_cand,
                                cudaStream_t st) {
  const int words = (c->n_orders + 31) >> 5;
  const size_t smem = (size_t)words * 4;
  cudaError_t e = cudaFuncSetAttribute(whp_validate_kernel,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       c->smem_optin - 1024);  // constant: see whp_swaps.cu
  if (e != cudaSuccess) return e;
  int64_t blocks = n_cand < (int64_t)c->num_sms * 8 ? n_cand : (int64_t)c->num_sms * 8;
  whp_validate_kernel<<<(unsigned)blocks, 256, smem, st>>>(d_perms, n_cand, c->n_orders,
                                                           c->d_count);
  c->launches += 1;
  return cudaGetLastError();
}
