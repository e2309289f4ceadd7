// whp_swaps.cu — whp_eval_swaps (a6, D8): pairwise-swap neighbourhood of a base plan with
// rescoring limited to the batches a swap can affect.
//
//   base pass   one walk of the base plan that tabulates, per batch b: first position
//               bstart[b], exclusive prefix of S-shape lengths bdist[b], class mask bclass[b];
//               plus batch_of_pos, base responses and totals.
//   neighbours  one warp per swap (i,j): batches before the one holding position i are
//               untouched (next-fit only looks forward) — except that when i opens its batch a
//               smaller order may slip into the previous cart, so the rewalk then starts one
//               batch earlier. The rewalk stops at the first new batch start P > j that is
//               also a base batch start (from there on both plans are identical), or at the
//               end. D and r are patched: minus the replaced base batches, plus the new ones.
#include "whp_walk.cuh"

namespace {

struct base_sink {
  whp_base_tables B;
  __device__ __forceinline__ void operator()(int32_t b, int32_t start_pos, int64_t dist,
                                             const uint32_t* cmask) {
    const int lane = whp_lane();
    if (lane == 0) { B.bstart[b] = start_pos; B.bdist[b] = dist; }
    if (lane < 8) B.bclass[(int64_t)b * 8 + lane] = cmask[lane];
  }
};

__global__ void __launch_bounds__(32)
whp_swaps_base_kernel(const whp_tables T, const int32_t* __restrict__ base_perm,
                      const whp_base_tables B) {
  __shared__ whp_warp_smem sm;
  const int lane = threadIdx.x;
  sm.amask[lane] = 0;
  if (lane < 8) sm.cmask[lane] = 0;
  for (int k = lane; k < T.K; k += 32) sm.r[k] = 0;
  __syncwarp();
  whp_walk_state st;
  whp_walk_init(st, 0);
  auto perm_at = [base_perm](int32_t p) { return __ldg(base_perm + p); };
  base_sink sink{B};
  whp_walk<false, false>(T, &sm, st, perm_at, 0, T.n_orders, whp_no_stop(), sink, B.bop);
  __syncwarp();
  const int32_t nb = st.b + 1;
  // exclusive prefix sum of the per-batch lengths, in place; bdist[nb] = D_base
  int64_t carry = 0;
  for (int32_t base = 0; base <= nb; base += 32) {
    const int32_t b = base + lane;
    const int64_t x = (b < nb) ? B.bdist[b] : 0;
    int64_t incl = x;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int64_t y = __shfl_up_sync(WHP_FULL, incl, d);
      if (lane >= d) incl += y;
    }
    if (b <= nb) B.bdist[b] = carry + incl - x;
    carry += __shfl_sync(WHP_FULL, incl, 31);
  }
  for (int k = lane; k < T.K; k += 32) B.resp[k] = sm.r[k];
  if (lane == 0) { B.bstart[nb] = T.n_orders; B.totals[0] = st.D; B.totals[1] = nb; }
}

struct swap_stop {
  const int32_t* bop;
  int32_t pj;
  __device__ __forceinline__ bool operator()(int32_t P) const {
    return P > pj && __ldg(bop + P) != __ldg(bop + P - 1);
  }
};

constexpr int kSwapWarps = 8;

__global__ void __launch_bounds__(kSwapWarps * 32)
whp_swaps_kernel(const whp_tables T, const int32_t* __restrict__ base_perm,
                 const whp_base_tables B, int32_t win_start, int32_t W, int64_t n_nb,
                 int64_t* __restrict__ d_dist, double* __restrict__ d_obj) {
  __shared__ whp_warp_smem sm_all[kSwapWarps];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  whp_warp_smem* sm = &sm_all[warp];
  sm->amask[lane] = 0;
  if (lane < 8) sm->cmask[lane] = 0;
  const int32_t nb = (int32_t)B.totals[1];
  const int KW = (T.K + 31) >> 5;
  for (int64_t n = (int64_t)blockIdx.x * kSwapWarps + warp; n < n_nb;
       n += (int64_t)gridDim.x * kSwapWarps) {
    // neighbour index -> (i', j'), row i' starts at i'(2W-i'-1)/2
    const double wm = 2.0 * W - 1.0;
    int64_t i = (int64_t)floor((wm - sqrt(wm * wm - 8.0 * (double)n)) * 0.5);
    i = max((int64_t)0, min(i, (int64_t)W - 2));
    while (i > 0 && i * (2 * (int64_t)W - i - 1) / 2 > n) --i;
    while ((i + 1) * (2 * (int64_t)W - i - 2) / 2 <= n) ++i;
    const int64_t j = i + 1 + (n - i * (2 * (int64_t)W - i - 1) / 2);
    const int32_t pi = win_start + (int32_t)i, pj = win_start + (int32_t)j;

    int32_t b0 = __ldg(B.bop + pi);
    int32_t p0 = __ldg(B.bstart + b0);
    if (pi == p0 && b0 > 0) { b0 -= 1; p0 = __ldg(B.bstart + b0); }
    for (int k = lane; k < T.K; k += 32) sm->r[k] = 0;
    __syncwarp();
    whp_walk_state st;
    whp_walk_init(st, b0);
    auto perm_at = [base_perm, pi, pj](int32_t p) {
      return __ldg(base_perm + (p == pi ? pj : (p == pj ? pi : p)));
    };
    const int32_t end = whp_walk<false, true>(T, sm, st, perm_at, p0, T.n_orders,
                                              swap_stop{B.bop, pj}, whp_no_sink(), nullptr);
    __syncwarp();
    const int32_t b_end = (end >= T.n_orders) ? nb : __ldg(B.bop + end);
    const int64_t D = B.totals[0] - (B.bdist[b_end] - B.bdist[b0]) + st.D;
    // r = r_base - (classes of the replaced base batches) + (classes of the new batches)
    for (int w = 0; w < KW; ++w) {
      const int k = 32 * w + lane;
      int32_t rk = (k < T.K) ? __ldg(B.resp + k) + sm->r[k] : 0;
      for (int32_t b = b0; b < b_end; ++b)
        rk -= (int32_t)((__ldg(B.bclass + (int64_t)b * 8 + w) >> lane) & 1u);
      if (k < T.K) sm->r[k] = rk;
    }
    __syncwarp();
    const double phi = whp_penalty(T, sm->r);
    if (lane == 0) {
      if (d_dist) d_dist[n] = D;
      if (d_obj) d_obj[n] = __dadd_rn((double)D, phi);
    }
    __syncwarp();
  }
}

}  // namespace

cudaError_t whp_launch_swaps(whp_ctx* c, const int32_t* d_base_perm, int32_t win_start,
                             int32_t win_len, int64_t* d_dist, double* d_obj, cudaStream_t st) {
  const whp_tables T = whp_make_tables(c);
  whp_swaps_base_kernel<<<1, 32, 0, st>>>(T, d_base_perm, c->base);
  c->launches += 1;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const int64_t n_nb = (int64_t)win_len * (win_len - 1) / 2;
  int64_t blocks = (n_nb + kSwapWarps - 1) / kSwapWarps;
  const int64_t cap = (int64_t)c->num_sms * 64;
  if (blocks > cap) blocks = cap;
  whp_swaps_kernel<<<(unsigned)blocks, kSwapWarps * 32, 0, st>>>(T, d_base_perm, c->base,
                                                                 win_start, win_len, n_nb,
                                                                 d_dist, d_obj);
  c->launches += 1;
  return cudaGetLastError();
}
