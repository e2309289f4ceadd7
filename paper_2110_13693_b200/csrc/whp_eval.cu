// whp_eval.cu — whp_eval_candidates: a1–a5 for explicit candidate plans.
// General kernel: one warp per candidate over the general walker (whp_walk.cuh); supports
// every output and any geometry within the limits.
#include <cstdlib>

#include "whp_walk.cuh"

namespace {

constexpr int kWarpsPerBlock = 8;

// DISTINCT: also count the distinct locations of every batch (n_distinct, D3) — a scan that is
// quadratic in the batch size, so it is compiled in only when that output is asked for.
template <bool DISTINCT>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
whp_eval_general_kernel(const whp_tables T, const int32_t* __restrict__ perms, int64_t n_cand,
                        const whp_eval_out out) {
  __shared__ whp_warp_smem sm_all[kWarpsPerBlock];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  whp_warp_smem* sm = &sm_all[warp];
  sm->amask[lane] = 0;
  if (lane < 8) sm->cmask[lane] = 0;
  for (int64_t cand = (int64_t)blockIdx.x * kWarpsPerBlock + warp; cand < n_cand;
       cand += (int64_t)gridDim.x * kWarpsPerBlock) {
    for (int k = lane; k < T.K; k += 32) sm->r[k] = 0;
    __syncwarp();
    const int32_t* row = perms + cand * T.n_orders;
    whp_walk_state st;
    whp_walk_init(st, 0);
    auto perm_at = [row](int32_t p) { return __ldg(row + p); };
    int32_t* bop_row = out.batch_of_pos ? out.batch_of_pos + cand * T.n_orders : nullptr;
    whp_walk<DISTINCT, false>(T, sm, st, perm_at, 0, T.n_orders, whp_no_stop(), whp_no_sink(),
                              bop_row);
    __syncwarp();
    const double phi = whp_penalty(T, sm->r);
    if (DISTINCT) {
      const int nd = __reduce_add_sync(WHP_FULL, st.n_distinct);
      if (lane == 0 && out.n_distinct) out.n_distinct[cand] = nd;
    }
    if (out.resp)
      for (int k = lane; k < T.K; k += 32) out.resp[cand * T.K + k] = sm->r[k];
    if (lane == 0) {
      if (out.dist) out.dist[cand] = st.D;
      if (out.penalty) out.penalty[cand] = phi;
      if (out.obj) out.obj[cand] = __dadd_rn((double)st.D, phi);
      if (out.n_batches) out.n_batches[cand] = st.b + 1;
      if (out.batch_hash) out.batch_hash[cand] = st.hash;
    }
    __syncwarp();
  }
}

}  // namespace

cudaError_t whp_launch_eval(whp_ctx* c, const int32_t* d_perms, int64_t n_cand,
                            const whp_eval_out& out, cudaStream_t st) {
  const whp_tables T = whp_make_tables(c);
  const bool detail = out.n_distinct != nullptr;  // only the general walker counts distinct locations
  if (!detail && whp_fast_eligible(c) && !c->dbg_force_general)
    return whp_launch_eval_fast(c, d_perms, n_cand, out, st);
  int64_t blocks = (n_cand + kWarpsPerBlock - 1) / kWarpsPerBlock;
  const int64_t cap = (int64_t)c->num_sms * 64;
  if (blocks > cap) blocks = cap;
  if (detail)
    whp_eval_general_kernel<true><<<(unsigned)blocks, kWarpsPerBlock * 32, 0, st>>>(
        T, d_perms, n_cand, out);
  else
    whp_eval_general_kernel<false><<<(unsigned)blocks, kWarpsPerBlock * 32, 0, st>>>(
        T, d_perms, n_cand, out);
  c->launches += 1;
  return cudaGetLastError();
}
