// whp_nhatc.cu — NEXT-1: the NHATC outer loop around the subsystem solve, on the device.
// PAPER.md:152-162 (§5, Eq. 3): subproblems exchange targets t and responses r and minimise
// f + phi(c); the update of phi's parameters is not printed (the paper cites Tosserams et al.
// 2010). DESIGN.md reading N1: v <- v + 2 w^2 c, w <- beta w, c = t - r*, with
// r* the responses of the plan the solve returned. Rounding order (shared by spec with the
// oracle): u = w*w; g = u*c; v' = v + 2*g; w' = beta*w.
#include "whp_internal.cuh"

namespace {

__global__ void whp_nhatc_update_kernel(double* __restrict__ tvw, int32_t K,
                                        const int32_t* __restrict__ resp_rows,
                                        const int64_t* __restrict__ d_idx, double beta) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= K) return;
  const int64_t row = d_idx ? *d_idx : 0;
  const double c = __dsub_rn(tvw[k], (double)resp_rows[row * K + k]);
  const double w = tvw[2 * K + k];
  const double u = __dmul_rn(w, w);
  const double g = __dmul_rn(u, c);
  tvw[K + k] = __dadd_rn(tvw[K + k], __dmul_rn(2.0, g));
  tvw[2 * K + k] = __dmul_rn(beta, w);
}

// history of one outer iteration: winner, its D and J
__global__ void whp_nhatc_record_kernel(const int64_t* __restrict__ d_idx,
                                        const int64_t* __restrict__ dist,
                                        const double* __restrict__ obj, int32_t it,
                                        int64_t* __restrict__ idx_hist,
                                        int64_t* __restrict__ dist_hist,
                                        double* __restrict__ obj_hist) {
  const int64_t i = *d_idx;
  if (idx_hist) idx_hist[it] = i;
  if (dist_hist) dist_hist[it] = dist[i];
  if (obj_hist) obj_hist[it] = obj[i];
}

// D and r_k of a plan do not depend on (t, v, w): inside one whp_nhatc_solve call the plans are
// evaluated once, and every later outer iteration only redoes D6 on the stored response rows —
// one warp per plan, the canonical accumulation (lane l adds its classes l, l+32, ... in
// ascending order, then the xor butterfly), so phi and J have the bits a full evaluation gives.
__global__ void __launch_bounds__(256)
whp_nhatc_rescore_kernel(const double* __restrict__ tvw, int32_t K,
                         const int32_t* __restrict__ resp_rows, const int64_t* __restrict__ dist,
                         int64_t n_cand, double* __restrict__ obj) {
  const int lane = threadIdx.x & 31;
  const int64_t cand = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (cand >= n_cand) return;
  const int32_t* __restrict__ row = resp_rows + cand * K;
  double phi = 0.0;
  for (int k = lane; k < K; k += 32) {
    const double c = __dsub_rn(tvw[k], (double)row[k]);
    const double u = __dmul_rn(tvw[2 * K + k], c);
    phi = __dadd_rn(phi, __dadd_rn(__dmul_rn(tvw[K + k], c), __dmul_rn(u, u)));
  }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) phi = __dadd_rn(phi, __shfl_xor_sync(0xffffffffu, phi, off));
  if (lane == 0) obj[cand] = __dadd_rn((double)dist[cand], phi);
}

}  // namespace

cudaError_t whp_launch_nhatc_rescore(whp_ctx* c, const int32_t* d_resp_rows, const int64_t* d_dist,
                                     int64_t n_cand, double* d_obj, cudaStream_t st) {
  const int64_t blocks = (n_cand * 32 + 255) / 256;
  whp_nhatc_rescore_kernel<<<(unsigned)blocks, 256, 0, st>>>(c->d_tvw, c->K, d_resp_rows, d_dist,
                                                             n_cand, d_obj);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t whp_launch_nhatc_update(whp_ctx* c, const int32_t* d_resp_rows, const int64_t* d_idx,
                                    double beta, cudaStream_t st) {
  whp_nhatc_update_kernel<<<(c->K + 127) / 128, 128, 0, st>>>(c->d_tvw, c->K, d_resp_rows, d_idx,
                                                              beta);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t whp_launch_nhatc_record(whp_ctx* c, const int64_t* d_idx, const int64_t* dist,
                                    const double* obj, int32_t it, int64_t* idx_hist,
                                    int64_t* dist_hist, double* obj_hist, cudaStream_t st) {
  whp_nhatc_record_kernel<<<1, 1, 0, st>>>(d_idx, dist, obj, it, idx_hist, dist_hist, obj_hist);
  c->launches += 1;
  return cudaGetLastError();
}
