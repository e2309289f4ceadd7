// whp_kmeans.cu — NEXT-3: subproblem 3, product placement by picking frequency with K-means.
// PAPER.md:134 (§5): "organize the products' positions concerning how often the products are
// selected ... using, e.g. K-means clustering". DESIGN.md reading N3 fixes the rest:
//   f_s = items of the day's orders that pick SKU s; c_j = lo + (j + 0.5) * ((hi - lo) / k);
//   iters x { nearest centroid (ties: lowest j); centroid = exact integer sum / count, one fp64
//   division; an empty cluster keeps its centroid }, a final assignment; clusters ranked by
//   centroid (largest first), SKUs ordered by (cluster rank, id), locations by
//   (|aisle - depot aisle|, aisle, slot, side); class = cluster * Z + slot * Z div S.
// Every step is a kernel; sums are integers (exact, order-free), so the result is bit-identical
// to the oracle's. The stable sort of the SKUs by cluster rank is cub::DeviceRadixSort.
#include <cub/device/device_radix_sort.cuh>

#include <vector>

#include "whp_internal.cuh"

namespace {

constexpr int kMaxK = 1024;

__global__ void km_freq_kernel(const int32_t* __restrict__ item_sku, int32_t n_items,
                               unsigned long long* __restrict__ freq) {
  for (int32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_items; i += gridDim.x * blockDim.x)
    atomicAdd(freq + item_sku[i], 1ull);
}

// min / max of the frequencies (two-value block reduction, then atomics)
__global__ void km_range_kernel(const unsigned long long* __restrict__ freq, int32_t n_skus,
                                unsigned long long* __restrict__ lohi) {
  unsigned long long lo = ~0ull, hi = 0ull;
  for (int32_t s = blockIdx.x * blockDim.x + threadIdx.x; s < n_skus; s += gridDim.x * blockDim.x) {
    const unsigned long long f = freq[s];
    lo = f < lo ? f : lo;
    hi = f > hi ? f : hi;
  }
  for (int o = 16; o >= 1; o >>= 1) {
    const unsigned long long l2 = __shfl_xor_sync(0xffffffffu, lo, o), h2 = __shfl_xor_sync(0xffffffffu, hi, o);
    lo = l2 < lo ? l2 : lo;
    hi = h2 > hi ? h2 : hi;
  }
  if ((threadIdx.x & 31) == 0) { atomicMin(lohi, lo); atomicMax(lohi + 1, hi); }
}

__global__ void km_init_kernel(const unsigned long long* __restrict__ lohi, int32_t k,
                               double* __restrict__ cent) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= k) return;
  const double lo = (double)lohi[0];
  const double step = __ddiv_rn((double)(lohi[1] - lohi[0]), (double)k);
  cent[j] = __dadd_rn(lo, __dmul_rn(__dadd_rn((double)j, 0.5), step));
}

// nearest centroid of every SKU (ties: lowest index); optionally accumulate the clusters' integer
// sums and counts (shared-memory privatised)
__global__ void km_assign_kernel(const unsigned long long* __restrict__ freq, int32_t n_skus,
                                 const double* __restrict__ cent, int32_t k,
                                 int32_t* __restrict__ assign, unsigned long long* __restrict__ sums,
                                 unsigned long long* __restrict__ cnts) {
  __shared__ double s_c[kMaxK];
  __shared__ unsigned long long s_sum[kMaxK], s_cnt[kMaxK];
  for (int j = threadIdx.x; j < k; j += blockDim.x) { s_c[j] = cent[j]; s_sum[j] = 0; s_cnt[j] = 0; }
  __syncthreads();
  for (int32_t s = blockIdx.x * blockDim.x + threadIdx.x; s < n_skus; s += gridDim.x * blockDim.x) {
    const double f = (double)freq[s];
    int best = 0;
    double bd = fabs(__dsub_rn(f, s_c[0]));
    for (int j = 1; j < k; ++j) {
      const double d = fabs(__dsub_rn(f, s_c[j]));
      if (d < bd) { bd = d; best = j; }
    }
    assign[s] = best;
    if (sums) { atomicAdd(&s_sum[best], freq[s]); atomicAdd(&s_cnt[best], 1ull); }
  }
  if (!sums) return;
  __syncthreads();
  for (int j = threadIdx.x; j < k; j += blockDim.x)
    if (s_cnt[j]) { atomicAdd(sums + j, s_sum[j]); atomicAdd(cnts + j, s_cnt[j]); }
}

__global__ void km_update_kernel(double* __restrict__ cent, int32_t k,
                                 unsigned long long* __restrict__ sums,
                                 unsigned long long* __restrict__ cnts) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= k) return;
  if (cnts[j]) cent[j] = __ddiv_rn((double)sums[j], (double)cnts[j]);
  sums[j] = 0;
  cnts[j] = 0;
}

// rank of a cluster: larger centroid first, ties to the lower index; rank of an aisle by
// (|a - a0|, a); sort key of a SKU = rank of its cluster
__global__ void km_ranks_kernel(const double* __restrict__ cent, int32_t k, int32_t* __restrict__ crank,
                                int32_t n_aisles, int32_t depot, int32_t* __restrict__ aisle_at) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < k) {
    int r = 0;
    for (int i = 0; i < k; ++i) r += cent[i] > cent[t] || (cent[i] == cent[t] && i < t);
    crank[t] = r;
  }
  if (t < n_aisles) {
    const int d = abs(t - depot);
    int r = 0;
    for (int a = 0; a < n_aisles; ++a) {
      const int da = abs(a - depot);
      r += da < d || (da == d && a < t);
    }
    aisle_at[r] = t;
  }
}

__global__ void km_keys_kernel(const int32_t* __restrict__ assign, const int32_t* __restrict__ crank,
                               int32_t n_skus, uint32_t* __restrict__ keys, int32_t* __restrict__ ids) {
  const int32_t s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n_skus) return;
  keys[s] = (uint32_t)crank[assign[s]];
  ids[s] = s;
}

__global__ void km_place_kernel(const int32_t* __restrict__ sorted_ids, const int32_t* __restrict__ assign,
                                const int32_t* __restrict__ aisle_at, int32_t n_skus, int32_t S,
                                int32_t Z, int32_t* __restrict__ sku_loc, int32_t* __restrict__ sku_class) {
  const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_skus) return;
  const int32_t s = sorted_ids[i];
  const int32_t a = aisle_at[i / (2 * S)], rem = i % (2 * S);
  const int32_t slot = rem / 2, side = rem % 2;
  sku_loc[s] = a * 2 * S + side * S + slot;
  sku_class[s] = assign[s] * Z + (int32_t)((int64_t)slot * Z / S);
}

}  // namespace

extern "C" whp_status whp_kmeans_slotting(int32_t n_aisles, int32_t slots_per_side,
                                          int32_t depot_aisle, int32_t n_skus,
                                          const int32_t* item_sku, int32_t n_items, int32_t k,
                                          int32_t n_zones, int32_t iters, int32_t cuda_device,
                                          int32_t* sku_loc, int32_t* sku_class, int32_t* assign,
                                          double* centroids) {
  if (!item_sku || !sku_loc || !sku_class) return WHP_ERR_INVALID_ARG;
  if (n_aisles < 1 || slots_per_side < 1 || n_skus < 1 || n_items < 1 || k < 1 || n_zones < 1 ||
      iters < 0 || cuda_device < 0)
    return WHP_ERR_INVALID_ARG;
  if (n_aisles > WHP_MAX_AISLES || slots_per_side > WHP_MAX_SLOTS || k > kMaxK ||
      depot_aisle < 0 || depot_aisle >= n_aisles || (int64_t)n_skus > 2ll * n_aisles * slots_per_side ||
      (int64_t)k * n_zones > WHP_MAX_CLASSES)
    return WHP_ERR_OUT_OF_RANGE;
  for (int32_t i = 0; i < n_items; ++i)
    if (item_sku[i] < 0 || item_sku[i] >= n_skus) return WHP_ERR_OUT_OF_RANGE;
  int prev = -1;
  cudaGetDevice(&prev);
  if (cudaSetDevice(cuda_device) != cudaSuccess) return WHP_ERR_CUDA;
  // device scratch
  int32_t *d_items = nullptr, *d_assign = nullptr, *d_crank = nullptr, *d_aisle = nullptr,
          *d_ids = nullptr, *d_ids2 = nullptr, *d_loc = nullptr, *d_cls = nullptr;
  uint32_t *d_keys = nullptr, *d_keys2 = nullptr;
  unsigned long long *d_freq = nullptr, *d_lohi = nullptr, *d_sums = nullptr, *d_cnts = nullptr;
  double* d_cent = nullptr;
  void* d_tmp = nullptr;
  size_t tmp_bytes = 0;
  whp_status st = WHP_OK;
  cudaError_t e = cudaSuccess;
  auto A = [&](void** p, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(p, bytes); };
  A((void**)&d_items, 4 * (size_t)n_items); A((void**)&d_assign, 4 * (size_t)n_skus);
  A((void**)&d_crank, 4 * (size_t)k); A((void**)&d_aisle, 4 * (size_t)n_aisles);
  A((void**)&d_ids, 4 * (size_t)n_skus); A((void**)&d_ids2, 4 * (size_t)n_skus);
  A((void**)&d_loc, 4 * (size_t)n_skus); A((void**)&d_cls, 4 * (size_t)n_skus);
  A((void**)&d_keys, 4 * (size_t)n_skus); A((void**)&d_keys2, 4 * (size_t)n_skus);
  A((void**)&d_freq, 8 * (size_t)n_skus); A((void**)&d_lohi, 16);
  A((void**)&d_sums, 8 * (size_t)k); A((void**)&d_cnts, 8 * (size_t)k); A((void**)&d_cent, 8 * (size_t)k);
  if (e == cudaSuccess)
    e = cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, d_keys, d_keys2, d_ids, d_ids2, n_skus);
  A(&d_tmp, tmp_bytes ? tmp_bytes : 16);
  if (e == cudaSuccess) {
    const unsigned long long lohi0[2] = {~0ull, 0ull};
    cudaMemcpy(d_items, item_sku, 4 * (size_t)n_items, cudaMemcpyHostToDevice);
    cudaMemset(d_freq, 0, 8 * (size_t)n_skus);
    cudaMemset(d_sums, 0, 8 * (size_t)k);
    cudaMemset(d_cnts, 0, 8 * (size_t)k);
    cudaMemcpy(d_lohi, lohi0, 16, cudaMemcpyHostToDevice);
    const int T = 256;
    const int gs = (n_skus + T - 1) / T < 1024 ? (n_skus + T - 1) / T : 1024;
    const int gi = (n_items + T - 1) / T < 1024 ? (n_items + T - 1) / T : 1024;
    km_freq_kernel<<<gi, T>>>(d_items, n_items, d_freq);
    km_range_kernel<<<gs, T>>>(d_freq, n_skus, d_lohi);
    km_init_kernel<<<(k + T - 1) / T, T>>>(d_lohi, k, d_cent);
    for (int32_t it = 0; it < iters; ++it) {
      km_assign_kernel<<<gs, T>>>(d_freq, n_skus, d_cent, k, d_assign, d_sums, d_cnts);
      km_update_kernel<<<(k + T - 1) / T, T>>>(d_cent, k, d_sums, d_cnts);
    }
    km_assign_kernel<<<gs, T>>>(d_freq, n_skus, d_cent, k, d_assign, nullptr, nullptr);
    const int nr = k > n_aisles ? k : n_aisles;
    km_ranks_kernel<<<(nr + T - 1) / T, T>>>(d_cent, k, d_crank, n_aisles, depot_aisle, d_aisle);
    km_keys_kernel<<<(n_skus + T - 1) / T, T>>>(d_assign, d_crank, n_skus, d_keys, d_ids);
    cub::DeviceRadixSort::SortPairs(d_tmp, tmp_bytes, d_keys, d_keys2, d_ids, d_ids2, n_skus);
    km_place_kernel<<<(n_skus + T - 1) / T, T>>>(d_ids2, d_assign, d_aisle, n_skus, slots_per_side,
                                                 n_zones, d_loc, d_cls);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpy(sku_loc, d_loc, 4 * (size_t)n_skus, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(sku_class, d_cls, 4 * (size_t)n_skus, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && assign) e = cudaMemcpy(assign, d_assign, 4 * (size_t)n_skus, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && centroids) e = cudaMemcpy(centroids, d_cent, 8 * (size_t)k, cudaMemcpyDeviceToHost);
  }
  if (e != cudaSuccess) st = e == cudaErrorMemoryAllocation ? WHP_ERR_NOMEM : WHP_ERR_CUDA;
  cudaFree(d_items); cudaFree(d_assign); cudaFree(d_crank); cudaFree(d_aisle); cudaFree(d_ids);
  cudaFree(d_ids2); cudaFree(d_loc); cudaFree(d_cls); cudaFree(d_keys); cudaFree(d_keys2);
  cudaFree(d_freq); cudaFree(d_lohi); cudaFree(d_sums); cudaFree(d_cnts); cudaFree(d_cent);
  cudaFree(d_tmp);
  if (prev >= 0) cudaSetDevice(prev);
  return st;
}
