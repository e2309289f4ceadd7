// whp_walk.cuh — the general warp walker: one warp walks a range of positions of one plan,
// 32 positions per tile, and performs a2–a5 of the hot path:
//   next-fit batching (D2) by a warp prefix sum + boundary chase,
//   per-batch aisle / class occupancy bitmasks in shared memory (D3),
//   S-shape length per batch from popc / max reductions, int64 (D4),
//   class-visit counters r_k (D5).
// It is the reference-quality device path: every feature (detail outputs, per-batch sinks,
// early stop for the swap evaluator, any geometry within the limits). The tuned candidate
// kernel in whp_eval.cu is a specialisation that must agree with it bit for bit.
#pragma once
#include "whp_internal.cuh"

#define WHP_FULL 0xffffffffu

struct whp_warp_smem {
  uint32_t amask[32];           // aisle occupancy of the open batch, word w owned by lane w
  uint32_t cmask[8];            // class occupancy of the open batch
  int32_t r[WHP_MAX_CLASSES];   // responses r_k of the plan being walked
};

struct whp_walk_state {  // warp-uniform
  int32_t load;       // items in the open batch (0: none open)
  int32_t b;          // index of the open batch, -1 before the first
  int32_t start_pos;  // first position of the open batch
  uint32_t kmax;      // max pick record of the open batch -> (a_max, deepest slot there)
  int64_t D;          // Σ dist_b of closed batches
  uint64_t hash;      // Σ (start_pos_b+1)(2b+1)
  int32_t n_distinct; // lane-local partial count (detail mode)
};

__device__ __forceinline__ void whp_walk_init(whp_walk_state& st, int32_t first_batch) {
  st.load = 0; st.b = first_batch - 1; st.start_pos = 0; st.kmax = 0;
  st.D = 0; st.hash = 0; st.n_distinct = 0;
}

__device__ __forceinline__ int whp_lane() { return threadIdx.x & 31; }

__device__ __forceinline__ int32_t whp_warp_incl_scan(int32_t x) {
  const int lane = whp_lane();
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    int32_t y = __shfl_up_sync(WHP_FULL, x, d);
    if (lane >= d) x += y;
  }
  return x;
}

// D4 for the open batch; clears its masks; adds its classes to r (D5). Warp-collective.
template <class BatchSink>
__device__ __forceinline__ void whp_close_batch(const whp_tables& T, whp_warp_smem* sm,
                                                whp_walk_state& st, BatchSink& sink) {
  const int lane = whp_lane();
  __syncwarp();
  const uint32_t aw = sm->amask[lane];
  sm->amask[lane] = 0;
  const int m = __reduce_add_sync(WHP_FULL, __popc(aw));
  const int lo = aw ? lane * 32 + __ffs(aw) - 1 : 0x7fffffff;
  const int64_t a_min = __reduce_min_sync(WHP_FULL, lo);
  const int64_t a_max = WHP_PICK_AISLE(st.kmax);
  const int64_t d_last =
      (int64_t)((st.kmax >> WHP_PICK_SLOT_SHIFT) & WHP_PICK_SLOT_MASK) * T.g.slot_pitch;
  const int64_t a0 = T.g.depot_aisle;
  const int64_t H = (int64_t)T.g.aisle_spacing *
                    (llabs(a0 - a_min) + (a_max - a_min) + llabs(a_max - a0));
  const int64_t Vt = (m & 1) ? (int64_t)(m - 1) * T.g.aisle_len + 2 * d_last
                             : (int64_t)m * T.g.aisle_len;
  const int64_t dist = H + Vt;
  st.D += dist;
  const int KW = (T.K + 31) >> 5;
  for (int w = 0; w < KW; ++w) {
    const uint32_t word = sm->cmask[w];
    if ((word >> lane) & 1u) sm->r[32 * w + lane] += 1;
  }
  sink(st.b, st.start_pos, dist, sm->cmask);
  __syncwarp();
  if (lane < 8) sm->cmask[lane] = 0;
  st.kmax = 0;
  __syncwarp();
}

struct whp_no_sink {
  __device__ __forceinline__ void operator()(int32_t, int32_t, int64_t, const uint32_t*) {}
};
struct whp_no_stop {
  __device__ __forceinline__ bool operator()(int32_t) const { return false; }
};

// Walk positions [p_begin, p_end) of the plan perm_at(.). Returns the position where the walk
// ended: p_end, or the first new-batch start P for which stop_at(P) was true (that batch is
// not opened). The last open batch is closed before returning.
template <bool DETAIL, bool CAN_STOP, class PermAt, class StopAt, class BatchSink>
__device__ __forceinline__ int32_t whp_walk(const whp_tables& T, whp_warp_smem* sm,
                                            whp_walk_state& st, PermAt perm_at, int32_t p_begin,
                                            int32_t p_end, StopAt stop_at, BatchSink sink,
                                            int32_t* batch_of_pos_row) {
  const int lane = whp_lane();
  int32_t end_pos = p_end;
  bool stopped = false;
  for (int32_t tile = p_begin; tile < p_end && !stopped; tile += 32) {
    const int32_t pos = tile + lane;
    int nvalid = min(32, p_end - tile);
    bool valid = lane < nvalid;
    uint32_t orec = 0;
    if (valid) orec = __ldg(T.order_rec + perm_at(pos));
    const int32_t q = valid ? (int32_t)(orec & WHP_Q_MASK) : 0;
    const int32_t off = (int32_t)(orec >> WHP_Q_BITS);
    const int32_t incl = whp_warp_incl_scan(q);
    const int32_t S = incl - q;
    // ---- D2: chase the batch boundaries inside this tile
    int32_t cur = -st.load;
    uint32_t starts = (st.load == 0) ? 1u : 0u;
    int from = (st.load == 0) ? 1 : 0;
    while (from < 32) {
      const uint32_t viol =
          __ballot_sync(WHP_FULL, valid && (incl - cur > T.C)) & (WHP_FULL << from);
      if (!viol) break;
      const int p = __ffs(viol) - 1;
      if (CAN_STOP && stop_at(tile + p)) {
        stopped = true; end_pos = tile + p; nvalid = p; valid = lane < nvalid;
        break;
      }
      starts |= 1u << p;
      cur = __shfl_sync(WHP_FULL, S, p);
      from = p + 1;
    }
    if (nvalid == 0) break;
    const int32_t b_tile = st.b;
    if (batch_of_pos_row != nullptr && valid)
      batch_of_pos_row[pos] = b_tile + __popc(starts & (WHP_FULL >> (31 - lane)));
    // ---- D3: per segment (= part of one batch inside this tile) fill the occupancy masks
    int lo = 0;
    while (lo < nvalid) {
      if ((starts >> lo) & 1u) {
        if (st.load > 0 || lo > 0) whp_close_batch(T, sm, st, sink);
        st.b += 1;
        st.start_pos = tile + lo;
        st.hash += (uint64_t)(st.start_pos + 1) * (uint64_t)(2 * (int64_t)st.b + 1);
      }
      const uint32_t rest = (lo + 1 < 32) ? (starts & (WHP_FULL << (lo + 1))) : 0u;
      const int hi = rest ? min(__ffs(rest) - 1, nvalid) : nvalid;
      uint32_t km = 0;
      if (lane >= lo && lane < hi) {
        for (int32_t i = 0; i < q; ++i) {
          const uint32_t pr = __ldg(T.pick_rec + off + i);
          km = max(km, pr);
          const uint32_t a = WHP_PICK_AISLE(pr);
          const uint32_t c = pr & WHP_PICK_CLASS_MASK;
          atomicOr(&sm->amask[a >> 5], 1u << (a & 31));
          atomicOr(&sm->cmask[c >> 5], 1u << (c & 31));
          if (DETAIL) {
            // |L_b| (D3): count this pick iff no earlier pick of the batch has its location
            bool dup = false;
            for (int32_t p2 = st.start_pos; p2 <= pos && !dup; ++p2) {
              const uint32_t o2 = __ldg(T.order_rec + perm_at(p2));
              const int32_t q2 = (p2 == pos) ? i : (int32_t)(o2 & WHP_Q_MASK);
              const int32_t off2 = (int32_t)(o2 >> WHP_Q_BITS);
              for (int32_t i2 = 0; i2 < q2; ++i2)
                if ((__ldg(T.pick_rec + off2 + i2) >> WHP_PICK_LOC_SHIFT) ==
                    (pr >> WHP_PICK_LOC_SHIFT)) { dup = true; break; }
            }
            if (!dup) st.n_distinct += 1;
          }
        }
      }
      st.kmax = max(st.kmax, __reduce_max_sync(WHP_FULL, km));
      lo = hi;
    }
    st.load = __shfl_sync(WHP_FULL, incl, nvalid - 1) - cur;
  }
  if (st.load > 0) {
    whp_close_batch(T, sm, st, sink);
    st.load = 0;
  }
  return end_pos;
}

// D6: canonical 32-lane sum of term_k = v_k c_k + (w_k c_k)^2, c = t_k - r_k; every product and
// sum individually rounded (no FMA contraction). Returns phi on every lane.
__device__ __forceinline__ double whp_penalty(const whp_tables& T, const int32_t* r) {
  const int lane = whp_lane();
  double s = 0.0;
  for (int k = lane; k < T.K; k += 32) {
    const double c = __dsub_rn(__ldg(T.tvw + k), (double)r[k]);
    const double u = __dmul_rn(__ldg(T.tvw + 2 * T.K + k), c);
    const double term = __dadd_rn(__dmul_rn(__ldg(T.tvw + T.K + k), c), __dmul_rn(u, u));
    s = __dadd_rn(s, term);
  }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) s = __dadd_rn(s, __shfl_xor_sync(WHP_FULL, s, off));
  return s;
}
