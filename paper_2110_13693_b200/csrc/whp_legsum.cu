// whp_legsum.cu — NEXT-2: the paper-literal subproblem 2. PAPER.md:125-129 (§5, Eq. 2):
// min sum d_i, d_i = shortest-path length between consecutive picking positions. DESIGN.md
// reading N2: every cart of the plan (next-fit, D2) leaves the depot, visits its picks in plan
// order and returns; a leg costs D0's walking metric, Dijkstra's closed form in this layout:
//   same aisle: |y1 - y2|;  else |a1 - a2| P + min(y1 + y2, 2A - y1 - y2).
// One warp per plan, 32 positions per tile: warp prefix sum of the item counts and a ballot-driven
// chase give the cart boundaries; a lane sums the legs inside its order and the leg that
// enters it (from the previous order's last pick, or from the depot when it opens a cart, plus
// the previous cart's way home); a shuffle reduction adds the lanes.
#include <cstdlib>

#include "whp_walk.cuh"

namespace {

struct pt { int32_t a; int64_t y; };

__device__ __forceinline__ pt pick_point(const whp_tables& T, uint32_t rec) {
  pt p;
  p.a = (int32_t)WHP_PICK_AISLE(rec);
  p.y = (int64_t)((rec >> WHP_PICK_SLOT_SHIFT) & WHP_PICK_SLOT_MASK) * T.g.slot_pitch;
  return p;
}
__device__ __forceinline__ int64_t leg(const whp_tables& T, pt u, pt v) {
  if (u.a == v.a) return llabs(u.y - v.y);
  const int64_t front = u.y + v.y, back = 2 * T.g.aisle_len - front;
  return llabs((int64_t)u.a - v.a) * T.g.aisle_spacing + (front < back ? front : back);
}

constexpr int kLegWarps = 8;

__global__ void __launch_bounds__(kLegWarps * 32)
whp_legsum_kernel(const whp_tables T, const int32_t* __restrict__ perms, int64_t n_cand,
                  int64_t* __restrict__ out_len) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const pt depot{T.g.depot_aisle, 0};
  for (int64_t cand = (int64_t)blockIdx.x * kLegWarps + warp; cand < n_cand;
       cand += (int64_t)gridDim.x * kLegWarps) {
    const int32_t* __restrict__ row = perms + cand * T.n_orders;
    int64_t total = 0;
    int32_t load = 0;          // items in the open cart (0: none open yet)
    uint32_t carry_last = 0;   // last pick record of the previous tile
    bool any = false;          // a cart is open
    for (int32_t tile = 0; tile < T.n_orders; tile += 32) {
      const int32_t pos = tile + lane;
      const int nvalid = min(32, T.n_orders - tile);
      const bool valid = lane < nvalid;
      uint32_t orec = 0;
      if (valid) orec = __ldg(T.order_rec + __ldg(row + pos));
      const int32_t q = valid ? (int32_t)(orec & WHP_Q_MASK) : 0;
      const int32_t off = (int32_t)(orec >> WHP_Q_BITS);
      const int32_t incl = whp_warp_incl_scan(q);
      const int32_t excl = incl - q;
      // D2: cart boundaries inside this tile
      int32_t cur = -load;
      uint32_t starts = (load == 0) ? 1u : 0u;
      int from = (load == 0) ? 1 : 0;
      while (from < 32) {
        const uint32_t viol =
            __ballot_sync(WHP_FULL, valid && (incl - cur > T.C)) & (WHP_FULL << from);
        if (!viol) break;
        const int p = __ffs(viol) - 1;
        starts |= 1u << p;
        cur = __shfl_sync(WHP_FULL, excl, p);
        from = p + 1;
      }
      load = __shfl_sync(WHP_FULL, incl, nvalid - 1) - cur;
      // legs of this lane's order
      uint32_t first = 0, last = 0;
      int64_t sum = 0;
      if (valid) {
        first = __ldg(T.pick_rec + off);
        last = first;
        pt u = pick_point(T, first);
        for (int32_t i = 1; i < q; ++i) {
          last = __ldg(T.pick_rec + off + i);
          const pt v = pick_point(T, last);
          sum += leg(T, u, v);
          u = v;
        }
      }
      uint32_t prev_last = __shfl_up_sync(WHP_FULL, last, 1);
      if (lane == 0) prev_last = carry_last;
      if (valid) {
        const pt f = pick_point(T, first);
        if ((starts >> lane) & 1u) {
          // this order opens a cart: the previous cart (if any) walks home, this one sets out
          if (any || lane > 0) sum += leg(T, pick_point(T, prev_last), depot);
          sum += leg(T, depot, f);
        } else {
          sum += leg(T, pick_point(T, prev_last), f);
        }
      }
      any = true;
      carry_last = __shfl_sync(WHP_FULL, last, nvalid - 1);
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) sum += __shfl_xor_sync(WHP_FULL, sum, o);
      total += sum;
    }
    if (any) total += leg(T, pick_point(T, carry_last), depot);
    if (lane == 0) out_len[cand] = total;
  }
}

}  // namespace

cudaError_t whp_launch_legsum(whp_ctx* c, const int32_t* d_perms, int64_t n_cand, int64_t* d_len,
                              cudaStream_t st) {
  if (whp_fast_eligible(c) && !c->dbg_force_general)  // shapes the tuned path covers
    return whp_launch_legsum_fast(c, d_perms, n_cand, d_len, st);
  const whp_tables T = whp_make_tables(c);
  int64_t blocks = (n_cand + kLegWarps - 1) / kLegWarps;
  const int64_t cap = (int64_t)c->num_sms * 64;
  if (blocks > cap) blocks = cap;
  whp_legsum_kernel<<<(unsigned)blocks, kLegWarps * 32, 0, st>>>(T, d_perms, n_cand, d_len);
  c->launches += 1;
  return cudaGetLastError();
}
