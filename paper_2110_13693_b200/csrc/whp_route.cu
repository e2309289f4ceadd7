// whp_route.cu — NEXT-2, second half: the carts of a plan routed by the return
// (reading N5) or the largest-gap (reading N6) heuristic instead of the S-shape of D4.
// PAPER.md:125-132 (§5 Eq. 2) states the objective (min sum of travelled distances over a
// picking sequence) and prints no routing rule; DESIGN.md §2 gives the readings.
//
// Both policies need more than the S-shape's (number of aisles, deepest pick of the last aisle):
// return needs the deepest pick of EVERY visited aisle, largest gap every distinct depth of every
// aisle strictly between the first and the last. The table kept per open cart is therefore the
// list of its picks' (aisle, depth) keys — at most C entries — sorted at the cart's close: when
// C <= 32 (every config of BASELINE.json but the stress one) the keys live one per lane in
// registers and a 32-lane bitonic network of shuffles sorts them (whp_route32_kernel); else the
// list sits in shared memory and a bitonic network runs over it (whp_route_kernel).
// In sorted order an aisle is a run of equal high bits; its deepest pick is the run's last key and
// its gaps are differences of neighbours.
//
// One warp per plan, 32 positions per tile: warp prefix sum of the item counts and the
// ballot-driven boundary chase of the general walker (D2); lanes append the picks of their orders
// to the cart's key list and OR their classes into the cart's class mask (D5); the canonical
// penalty of D6 at the end. Results are bit-identical to the oracle's orc_eval_routing.
#include "whp_walk.cuh"

namespace {

constexpr int kRouteWarps = 8;
constexpr uint32_t kPadKey = 0xffffffffu;

struct route_warp_smem {
  uint32_t cmask[8];
  int32_t r[WHP_MAX_CLASSES];
};

// ascending bitonic sort of one key per lane
__device__ __forceinline__ uint32_t sort32(uint32_t key) {
  const int lane = whp_lane();
#pragma unroll
  for (int k = 2; k <= 32; k <<= 1)
#pragma unroll
    for (int j = k >> 1; j > 0; j >>= 1) {
      const uint32_t other = __shfl_xor_sync(WHP_FULL, key, j);
      const bool up = (lane & k) == 0, lower = (lane & j) == 0;
      key = (lower == up) ? min(key, other) : max(key, other);
    }
  return key;
}

// ascending bitonic sort of keys[0..p2) in shared memory, p2 a power of two >= 64
__device__ __forceinline__ void sort_smem(uint32_t* keys, int p2) {
  const int lane = whp_lane();
  for (int k = 2; k <= p2; k <<= 1)
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int t = lane; t < (p2 >> 1); t += 32) {
        const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));  // the lower index of pair t
        const uint32_t a = keys[i], b = keys[i | j];
        const bool up = (i & k) == 0;
        if ((a > b) == up) { keys[i] = b; keys[i | j] = a; }
      }
      __syncwarp();
    }
}

// Length of the cart whose n sorted keys (aisle << 12 | slot1) sit in keys[0..n): warp-collective,
// returns the same value on every lane. POLICY 1 = return (N5), 2 = largest gap (N6).
template <int POLICY>
__device__ __forceinline__ int64_t cart_length(const whp_tables& T, const uint32_t* keys, int n) {
  const int lane = whp_lane();
  const int64_t A = T.g.aisle_len, pitch = T.g.slot_pitch;
  const int32_t a_min = (int32_t)(keys[0] >> 12), a_max = (int32_t)(keys[n - 1] >> 12);
  const int64_t a0 = T.g.depot_aisle;
  const int64_t H = (int64_t)T.g.aisle_spacing *
                    (llabs(a0 - a_min) + ((int64_t)a_max - a_min) + llabs((int64_t)a_max - a0));
  int64_t part = 0;
  if (POLICY == 1 || a_min == a_max) {
    // deepest pick of every visited aisle: the last key of every run
    for (int i = lane; i < n; i += 32) {
      const uint32_t k = keys[i];
      const bool last = (i + 1 == n) || ((keys[i + 1] >> 12) != (k >> 12));
      if (last) part += 2 * (int64_t)(k & 0xfffu) * pitch;
    }
  } else {
    // first and last visited aisle: traversed completely; every aisle in between: all of it but
    // its largest gap, walked twice. The lane that holds an aisle's first key scans the run.
    if (lane == 0) part = 2 * A;
    for (int i = lane; i < n; i += 32) {
      const uint32_t k = keys[i];
      const int32_t a = (int32_t)(k >> 12);
      const bool first = (i == 0) || ((int32_t)(keys[i - 1] >> 12) != a);
      if (first && a != a_min && a != a_max) {
        int64_t y = (int64_t)(k & 0xfffu) * pitch;
        int64_t gap = y;  // front cross-aisle to the shallowest pick
        int j = i + 1;
        while (j < n && (int32_t)(keys[j] >> 12) == a) {
          const int64_t y2 = (int64_t)(keys[j] & 0xfffu) * pitch;
          gap = max(gap, y2 - y);
          y = y2;
          ++j;
        }
        gap = max(gap, A - y);  // deepest pick to the back cross-aisle
        part += 2 * (A - gap);
      }
    }
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) part += __shfl_xor_sync(WHP_FULL, part, o);
  return H + part;
}

template <int POLICY, bool REG_SORT>
__global__ void __launch_bounds__(kRouteWarps * 32)
whp_route_kernel(const whp_tables T, const int32_t* __restrict__ perms, int64_t n_cand, int p2max,
                 int64_t* __restrict__ dist_out, double* __restrict__ obj_out) {
  extern __shared__ __align__(16) uint8_t route_smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  route_warp_smem* sm = reinterpret_cast<route_warp_smem*>(route_smem) + warp;
  uint32_t* keys = reinterpret_cast<uint32_t*>(route_smem + kRouteWarps * sizeof(route_warp_smem)) +
                   (size_t)warp * p2max;
  if (lane < 8) sm->cmask[lane] = 0;
  const int KW = (T.K + 31) >> 5;
  for (int64_t cand = (int64_t)blockIdx.x * kRouteWarps + warp; cand < n_cand;
       cand += (int64_t)gridDim.x * kRouteWarps) {
    for (int k = lane; k < T.K; k += 32) sm->r[k] = 0;
    __syncwarp();
    const int32_t* row = perms + cand * T.n_orders;
    int32_t load = 0;   // items in the open cart (0: none open)
    int32_t nkeys = 0;  // keys of the open cart already in the list (= load)
    int64_t D = 0;

    auto close_cart = [&]() {  // warp-collective: sort the list, add the cart's length and classes
      __syncwarp();
      const int n = nkeys;
      if (REG_SORT) {
        const uint32_t key = sort32(lane < n ? keys[lane] : kPadKey);
        __syncwarp();
        keys[lane] = key;
      } else {
        int p2 = 32;
        while (p2 < n) p2 <<= 1;
        for (int i = n + lane; i < p2; i += 32) keys[i] = kPadKey;
        __syncwarp();
        if (p2 == 32) {
          const uint32_t key = sort32(keys[lane]);
          __syncwarp();
          keys[lane] = key;
        } else {
          sort_smem(keys, p2);
        }
      }
      __syncwarp();
      D += cart_length<POLICY>(T, keys, n);
      for (int w = 0; w < KW; ++w)
        if ((sm->cmask[w] >> lane) & 1u) sm->r[32 * w + lane] += 1;
      __syncwarp();
      if (lane < 8) sm->cmask[lane] = 0;
      nkeys = 0;
      __syncwarp();
    };

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
      // D2: positions of this tile at which a new cart opens
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
      // the parts of this tile, each inside one cart: append their picks to the cart's list
      int lo = 0;
      while (lo < nvalid) {
        if ((starts >> lo) & 1u) {
          if (load > 0 || lo > 0) close_cart();
        }
        const uint32_t rest = (lo + 1 < 32) ? (starts & (WHP_FULL << (lo + 1))) : 0u;
        const int hi = rest ? min(__ffs(rest) - 1, nvalid) : nvalid;
        const int32_t excl_lo = __shfl_sync(WHP_FULL, excl, lo);
        const int32_t incl_hi = __shfl_sync(WHP_FULL, incl, hi - 1);
        if (lane >= lo && lane < hi) {
          const int32_t dst = nkeys + (excl - excl_lo);
          for (int32_t i = 0; i < q; ++i) {
            const uint32_t pr = __ldg(T.pick_rec + off + i);
            keys[dst + i] = pr >> WHP_PICK_SLOT_SHIFT;  // aisle << 12 | slot1
            const uint32_t c = pr & WHP_PICK_CLASS_MASK;
            atomicOr(&sm->cmask[c >> 5], 1u << (c & 31));
          }
        }
        nkeys += incl_hi - excl_lo;
        lo = hi;
      }
      load = nkeys;
    }
    if (load > 0) close_cart();
    __syncwarp();
    const double phi = whp_penalty(T, sm->r);
    if (lane == 0) {
      if (dist_out) dist_out[cand] = D;
      if (obj_out) obj_out[cand] = __dadd_rn((double)D, phi);
    }
    __syncwarp();
  }
}


// ---------------------------------------------------------------------- carts of up to 32 picks
// C <= 32 (every configuration of BASELINE.json but the stress one): the open cart's keys never
// leave the registers. A tile part's picks are flattened over the lanes (item i of the part
// belongs to the last position whose item prefix is <= i: a five-step search by shuffles, then
// one pick load per lane), lane t of the cart holds key t; at the close the 32-lane bitonic
// network sorts them, runs of equal aisles are found by comparing neighbours (shuffles), the
// largest gap of a run by a segmented max-scan, and the cart's distinct classes by match_any
// (one leader per class bumps r_k). No shared memory but the r_k counters.
// len_t: int32_t when every per-cart quantity provably fits 31 bits (host check), else int64_t.
template <int POLICY, typename len_t>
__global__ void __launch_bounds__(kRouteWarps * 32)
whp_route32_kernel(const whp_tables T, const int32_t* __restrict__ perms, int64_t n_cand,
                   int64_t* __restrict__ dist_out, double* __restrict__ obj_out) {
  __shared__ int32_t r_all[kRouteWarps][WHP_MAX_CLASSES];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int32_t* r = r_all[warp];
  const len_t A = (len_t)T.g.aisle_len, pitch = (len_t)T.g.slot_pitch;
  const int64_t a0 = T.g.depot_aisle;
  for (int64_t cand = (int64_t)blockIdx.x * kRouteWarps + warp; cand < n_cand;
       cand += (int64_t)gridDim.x * kRouteWarps) {
    for (int k = lane; k < T.K; k += 32) r[k] = 0;
    __syncwarp();
    const int32_t* row = perms + cand * T.n_orders;
    int32_t load = 0, nkeys = 0;
    uint32_t key = kPadKey, cls = 0;  // this lane's pick of the open cart (lane < nkeys)
    int64_t D = 0;

    auto close_cart = [&]() {
      __syncwarp();  // the previous cart's r_k updates (other lanes) are done
      const int n = nkeys;
      const bool mine = lane < n;
      // D5: one leader per distinct class of the cart
      const uint32_t act = __ballot_sync(WHP_FULL, mine);
      if (mine) {
        const uint32_t same = __match_any_sync(act, cls);
        if ((int)(__ffs(same) - 1) == lane) r[cls] += 1;
      }
      // D3 on sorted keys
      const uint32_t sk = sort32(key);
      const int32_t a = (int32_t)(sk >> 12);
      const len_t y = (len_t)(sk & 0xfffu) * pitch;
      const uint32_t up = __shfl_up_sync(WHP_FULL, sk, 1), dn = __shfl_down_sync(WHP_FULL, sk, 1);
      const bool first = mine && (lane == 0 || (int32_t)(up >> 12) != a);
      const bool last = mine && (lane == n - 1 || (int32_t)(dn >> 12) != a);
      const int32_t a_min = __shfl_sync(WHP_FULL, a, 0), a_max = __shfl_sync(WHP_FULL, a, n - 1);
      const int64_t H = (int64_t)T.g.aisle_spacing *
                        (llabs(a0 - a_min) + ((int64_t)a_max - a_min) + llabs((int64_t)a_max - a0));
      len_t part = 0;
      if (POLICY == 1 || a_min == a_max) {
        if (last) part = 2 * y;  // deepest pick of every visited aisle
      } else {
        // largest gap of every run: front cross-aisle -> first pick, between neighbours, and
        // (at the run's last key) deepest pick -> back cross-aisle; segmented max-scan
        const len_t yup = (len_t)(up & 0xfffu) * pitch;
        len_t g = mine ? (first ? y : y - yup) : 0;
        if (last) g = max(g, A - y);
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const len_t og = __shfl_up_sync(WHP_FULL, g, d);
          const int32_t oa = __shfl_up_sync(WHP_FULL, a, d);
          if (lane >= d && oa == a) g = max(g, og);
        }
        if (last && a != a_min && a != a_max) part = 2 * (A - g);
        if (lane == 0) part += 2 * A;  // first and last visited aisle, traversed completely
      }
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) part += __shfl_xor_sync(WHP_FULL, part, o);
      D += H + (int64_t)part;
      key = kPadKey;
      nkeys = 0;
    };

    for (int32_t tile = 0; tile < T.n_orders; tile += 32) {
      const int32_t pos = tile + lane;
      const int nvalid = min(32, T.n_orders - tile);
      const bool valid = lane < nvalid;
      uint32_t orec = 0;
      if (valid) orec = __ldg(T.order_rec + __ldg(row + pos));
      const int32_t q = valid ? (int32_t)(orec & WHP_Q_MASK) : 0;
      const int32_t incl = whp_warp_incl_scan(q);
      const int32_t excl = incl - q;
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
      int lo = 0;
      while (lo < nvalid) {
        if ((starts >> lo) & 1u) {
          if (load > 0 || lo > 0) close_cart();
        }
        const uint32_t rest = (lo + 1 < 32) ? (starts & (WHP_FULL << (lo + 1))) : 0u;
        const int hi = rest ? min(__ffs(rest) - 1, nvalid) : nvalid;
        const int32_t excl_lo = __shfl_sync(WHP_FULL, excl, lo);
        const int32_t items = __shfl_sync(WHP_FULL, incl, hi - 1) - excl_lo;
        // item i = lane - nkeys of this part: its position j in [lo, hi) is the last one with
        // excl_j - excl_lo <= i (excl ascends over the lanes)
        const int32_t i = lane - nkeys;
        int j = lo;
#pragma unroll
        for (int step = 16; step >= 1; step >>= 1) {
          const int jj = j + step;
          const int32_t e = __shfl_sync(WHP_FULL, excl, jj & 31);
          if (jj < hi && e - excl_lo <= i) j = jj;
        }
        const uint32_t orec_j = __shfl_sync(WHP_FULL, orec, j);
        const int32_t excl_j = __shfl_sync(WHP_FULL, excl, j);
        if (i >= 0 && i < items) {
          const uint32_t pr = __ldg(T.pick_rec + (orec_j >> WHP_Q_BITS) + (i - (excl_j - excl_lo)));
          key = pr >> WHP_PICK_SLOT_SHIFT;  // aisle << 12 | slot1
          cls = pr & WHP_PICK_CLASS_MASK;
        }
        nkeys += items;
        lo = hi;
      }
      load = nkeys;
    }
    if (load > 0) close_cart();
    __syncwarp();
    const double phi = whp_penalty(T, r);
    if (lane == 0) {
      if (dist_out) dist_out[cand] = D;
      if (obj_out) obj_out[cand] = __dadd_rn((double)D, phi);
    }
    __syncwarp();
  }
}

}  // namespace

cudaError_t whp_launch_route(whp_ctx* c, const int32_t* d_perms, int64_t n_cand, int32_t policy,
                             int64_t* d_dist, double* d_obj, cudaStream_t st) {
  const whp_tables T = whp_make_tables(c);
  int p2max = 32;
  while (p2max < c->C) p2max <<= 1;
  const bool reg_sort = c->C <= 32;
  const size_t smem = kRouteWarps * (sizeof(route_warp_smem) + 4 * (size_t)p2max);
  int64_t blocks = (n_cand + kRouteWarps - 1) / kRouteWarps;
  const int64_t cap = (int64_t)c->num_sms * 32;
  if (blocks > cap) blocks = cap;
#define WHP_LAUNCH_ROUTE(POL, REG)                                                               \
  do {                                                                                           \
    cudaError_t e_ = cudaFuncSetAttribute(whp_route_kernel<POL, REG>,                            \
                                          cudaFuncAttributeMaxDynamicSharedMemorySize,           \
                                          c->smem_optin - 1024);                                 \
    if (e_ != cudaSuccess) return e_;                                                            \
    whp_route_kernel<POL, REG><<<(unsigned)blocks, kRouteWarps * 32, smem, st>>>(                \
        T, d_perms, n_cand, p2max, d_dist, d_obj);                                               \
  } while (0)
  if (reg_sort && !c->dbg_force_general) {  // carts of up to 32 picks: keys stay in registers
    // a cart's vertical travel is at most 2 A per pick (+ 2 A): 32-bit lengths when that fits
    const bool fits32 = 68ll * c->g.aisle_len < (1ll << 31);
#define WHP_LAUNCH_ROUTE32(POL, LEN)                                                             \
  whp_route32_kernel<POL, LEN><<<(unsigned)blocks, kRouteWarps * 32, 0, st>>>(T, d_perms, n_cand, \
                                                                             d_dist, d_obj)
    if (policy == WHP_ROUTE_RETURN) {
      if (fits32) WHP_LAUNCH_ROUTE32(1, int32_t); else WHP_LAUNCH_ROUTE32(1, int64_t);
    } else {
      if (fits32) WHP_LAUNCH_ROUTE32(2, int32_t); else WHP_LAUNCH_ROUTE32(2, int64_t);
    }
#undef WHP_LAUNCH_ROUTE32
  } else if (policy == WHP_ROUTE_RETURN) {
    if (reg_sort) WHP_LAUNCH_ROUTE(1, true); else WHP_LAUNCH_ROUTE(1, false);
  } else {
    if (reg_sort) WHP_LAUNCH_ROUTE(2, true); else WHP_LAUNCH_ROUTE(2, false);
  }
#undef WHP_LAUNCH_ROUTE
  c->launches += 1;
  return cudaGetLastError();
}
