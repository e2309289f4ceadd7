// whp_swaps.cu — whp_eval_swaps (a6, D8): pairwise-swap neighbourhood of a base plan with
// rescoring limited to the batches a swap can affect.
//
//   tables      whp_swaps_base_kernel (one block): item-count prefix pre[p], order record per
//               position, nxt[p] = end of the batch that would open at p (binary search), and the
//               base batch starts: the plan is cut into segments of >= C positions, every
//               segment tabulates where a chain that enters it at its k-th position leaves it,
//               one thread composes the segments' entry points, one thread per segment marks
//               its boundaries, a block scan ranks them (bstart[b], bop[p]).
//               whp_swaps_prep_kernel (multi-block): the hypothetical batch [p, nxt[p]) of every
//               position of the window region and of every base batch start, one warp per batch
//               with its picks flattened over the lanes (dist_at[p], cls_at[p]).
//               whp_swaps_tail_kernel (one launch, two block roles): the second half of the base
//               pass — prefix of the base batch lengths bdist[b], class-count prefix rpre[b][k],
//               base D, phi, J — and, per region position a neighbour can ask for, the sums along
//               its chain p -> nxt[p] -> ... up to where it meets the base plan (dtail, rtail, bF).
//               prep and tail are programmatic dependents of their predecessor.
//   neighbours  one warp per swap (pi,pj). Next-fit only looks forward, so batches before the
//               one holding pi are untouched — except that when pi opens its batch a smaller
//               order may slip into the previous cart, so the rewalk then starts one batch
//               earlier. Equal item counts leave every boundary in place: only the two batches
//               holding pi and pj are rescored. Otherwise the plan is re-batched from there;
//               only the batches holding a swapped position are scored from their picks, the
//               stretch between pi and pj is a difference of two chain sums and everything
//               after pj one chain look-up. D and r are patched: minus the replaced base
//               batches (prefix differences), plus the new ones.
#include <cstdlib>

#include "whp_walk.cuh"

namespace {

// Programmatic dependent launch: the table kernels of one whp_eval_swaps / whp_eval_moves call
// depend on each other in a row (base -> prep -> tail). A kernel launched with launch_dependent()
// may become resident while its predecessor still runs; it must pass dep_wait() — which returns
// once the predecessor grid has completed and its writes are visible — before it touches anything
// the predecessor writes. The predecessor allows that early start with dep_trigger() (all of its
// blocks are resident or done by then, so the waiting blocks cannot starve it). Every thread of a
// dependent kernel calls dep_wait(), so completion stays transitive along the row.
// The neighbour kernel itself is launched normally: as a third dependent it saves another 2 us
// of the call alone (74.8 instead of 76.7 us at W = 256), but its 1184 blocks then sit resident
// and idle on every SM while the tables are built, and a candidate evaluation running on
// another stream loses 0.03 ms of a 0.43 ms step to that (profiles/r2_head.md).
__device__ __forceinline__ void dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void dep_trigger() { asm volatile("griddepcontrol.launch_dependents;"); }

template <class... KArgs, class... Args>
cudaError_t launch_dependent(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem,
                             cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(block);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// The base plan with positions pi and pj exchanged (pi = pj = -1: the base plan itself), seen
// through the base tables: pre = exclusive item-count prefix, orec = order record by position.
// A window [lo, lo+cnt) of both tables may be staged in shared memory.
struct swap_seq {
  const int32_t* pre;      // global tables (plain loads: the base pass writes them itself)
  const uint32_t* orec;
  const int32_t* s_pre;    // shared-memory copy of pre[lo .. lo+n_pre)
  const uint32_t* s_orec;  // shared-memory copy of orec[lo .. lo+n_orec)
  int32_t lo;
  uint32_t n_pre, n_orec;  // 0: nothing staged
  int32_t pi, pj, delta;   // delta = q(pj) - q(pi)
  __device__ __forceinline__ int32_t pre_base(int32_t p) const {
    const uint32_t k = (uint32_t)(p - lo);
    return k < n_pre ? s_pre[k] : pre[p];
  }
  __device__ __forceinline__ int32_t pre_at(int32_t p) const {
    return pre_base(p) + ((p > pi && p <= pj) ? delta : 0);
  }
  __device__ __forceinline__ uint32_t orec_at(int32_t p) const {
    const int32_t s = (p == pi) ? pj : ((p == pj) ? pi : p);
    const uint32_t k = (uint32_t)(s - lo);
    return k < n_orec ? s_orec[k] : orec[s];
  }
};

// NEXT-4 (reading N4): the base plan with the order at position pi taken out and put back at
// position pj; the orders in between shift by one. qi = item count of the moved order.
struct move_seq {
  const int32_t* pre;
  const uint32_t* orec;
  const int32_t* s_pre;
  const uint32_t* s_orec;
  int32_t lo;
  uint32_t n_pre, n_orec;
  int32_t pi, pj, qi;
  __device__ __forceinline__ int32_t pre_base(int32_t p) const {
    const uint32_t k = (uint32_t)(p - lo);
    return k < n_pre ? s_pre[k] : pre[p];
  }
  __device__ __forceinline__ int32_t pre_at(int32_t p) const {
    if (pi < pj) return (p > pi && p <= pj) ? pre_base(p + 1) - qi : pre_base(p);
    return (p > pj && p <= pi) ? pre_base(p - 1) + qi : pre_base(p);
  }
  __device__ __forceinline__ int32_t base_of(int32_t p) const {  // base position of new position p
    if (p == pj) return pi;
    if (pi < pj) return (p >= pi && p < pj) ? p + 1 : p;
    return (p > pj && p <= pi) ? p - 1 : p;
  }
  __device__ __forceinline__ uint32_t orec_at(int32_t p) const {
    const int32_t s = base_of(p);
    const uint32_t k = (uint32_t)(s - lo);
    return k < n_orec ? s_orec[k] : orec[s];
  }
};

struct warp_sets {
  uint32_t amask[32];  // aisle occupancy of the batch being scored
  uint32_t cmask[8];   // class occupancy
};

// End of the batch that opens at position p (D2): the largest e <= n with
// pre(e) - pre(p) <= C. Every order has at least one item, so e - p <= C. Warp-collective.
template <class Seq>
__device__ __forceinline__ int32_t batch_end(const Seq& q, int32_t p, int32_t n, int32_t C) {
  const int lane = whp_lane();
  const int32_t lim = q.pre_at(p) + C;
  int32_t e = p;
  for (;;) {
    const int32_t cand = e + 1 + lane;
    const bool ok = cand <= n && q.pre_at(cand) <= lim;
    const uint32_t bal = __ballot_sync(WHP_FULL, ok);
    const int cnt = (bal == WHP_FULL) ? 32 : __ffs(~bal) - 1;  // prefix is increasing
    e += cnt;
    if (cnt < 32) return e;
  }
}

// D3 + D4 of the batch at positions [s, e): the picks of the batch are flattened over the
// lanes (item t belongs to the last position whose prefix is <= t). Returns dist_b on every
// lane; leaves the batch's class mask in sets->cmask (the caller consumes and clears it).
template <class Seq>
__device__ __forceinline__ int64_t score_batch(const whp_tables& T, warp_sets* sets,
                                               const Seq& q, int32_t s, int32_t e) {
  const int lane = whp_lane();
  const int32_t base0 = q.pre_at(s);
  const int32_t load = q.pre_at(e) - base0;
  uint32_t kmax = 0, kmin = 0xffffffffu;
  const int32_t npos = e - s;
  if (npos <= 32) {
    // one position per lane: its relative prefix (ascending over the lanes) and order record;
    // an item finds its position by a binary search over the lanes (shuffles, no table access)
    const int32_t mine = lane < npos ? q.pre_at(s + lane) - base0 : 0x7fffffff;
    const uint32_t my_orec = lane < npos ? q.orec_at(s + lane) : 0u;
    for (int32_t t0 = 0; t0 < load; t0 += 32) {
      const int32_t t = t0 + lane;
      int l = 0;  // largest lane with mine <= t (mine of lane 0 is 0)
#pragma unroll
      for (int step = 16; step >= 1; step >>= 1) {
        const int32_t v = __shfl_sync(WHP_FULL, mine, (l + step) & 31);
        if (l + step < 32 && v <= t) l += step;
      }
      const uint32_t orec = __shfl_sync(WHP_FULL, my_orec, l);
      const int32_t first = __shfl_sync(WHP_FULL, mine, l);
      if (t < load) {
        const uint32_t pr = __ldg(T.pick_rec + (orec >> WHP_Q_BITS) + (t - first));
        kmax = max(kmax, pr);
        kmin = min(kmin, pr);
        const uint32_t a = WHP_PICK_AISLE(pr);
        const uint32_t c = pr & WHP_PICK_CLASS_MASK;
        atomicOr(&sets->amask[a >> 5], 1u << (a & 31));
        atomicOr(&sets->cmask[c >> 5], 1u << (c & 31));
      }
    }
  } else
  for (int32_t t0 = 0; t0 < load; t0 += 32) {
    const int32_t t = t0 + lane;
    if (t < load) {
      int32_t lo = s, hi = e - 1;
      while (lo < hi) {
        const int32_t mid = (lo + hi + 1) >> 1;
        if (q.pre_at(mid) - base0 <= t) lo = mid; else hi = mid - 1;
      }
      const uint32_t orec = q.orec_at(lo);
      const uint32_t pr = __ldg(T.pick_rec + (orec >> WHP_Q_BITS) + (t - (q.pre_at(lo) - base0)));
      kmax = max(kmax, pr);
      kmin = min(kmin, pr);
      const uint32_t a = WHP_PICK_AISLE(pr);
      const uint32_t c = pr & WHP_PICK_CLASS_MASK;
      atomicOr(&sets->amask[a >> 5], 1u << (a & 31));
      atomicOr(&sets->cmask[c >> 5], 1u << (c & 31));
    }
  }
  kmax = __reduce_max_sync(WHP_FULL, kmax);
  kmin = __reduce_min_sync(WHP_FULL, kmin);
  __syncwarp();
  const uint32_t aw = sets->amask[lane];
  sets->amask[lane] = 0;
  const int m = __reduce_add_sync(WHP_FULL, __popc(aw));
  const int64_t a_max = WHP_PICK_AISLE(kmax), a_min = WHP_PICK_AISLE(kmin);
  const int64_t d_last =
      (int64_t)((kmax >> WHP_PICK_SLOT_SHIFT) & WHP_PICK_SLOT_MASK) * T.g.slot_pitch;
  const int64_t a0 = T.g.depot_aisle;
  const int64_t H = (int64_t)T.g.aisle_spacing *
                    (llabs(a0 - a_min) + (a_max - a_min) + llabs(a_max - a0));
  const int64_t Vt = (m & 1) ? (int64_t)(m - 1) * T.g.aisle_len + 2 * d_last
                             : (int64_t)m * T.g.aisle_len;
  return H + Vt;
}

// D6 with lane l owning classes l, l+32, ... (the canonical 32-lane accumulation)
__device__ __forceinline__ double penalty_regs(const whp_tables& T, const int32_t (&r)[8]) {
  const int lane = whp_lane();
  double s = 0.0;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    const int k = 32 * w + lane;
    if (k < T.K) {
      const double c = __dsub_rn(__ldg(T.tvw + k), (double)r[w]);
      const double u = __dmul_rn(__ldg(T.tvw + 2 * T.K + k), c);
      const double term = __dadd_rn(__dmul_rn(__ldg(T.tvw + T.K + k), c), __dmul_rn(u, u));
      s = __dadd_rn(s, term);
    }
  }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) s = __dadd_rn(s, __shfl_xor_sync(WHP_FULL, s, off));
  return s;
}

// ------------------------------------------------------------------------------ base pass
constexpr int kBaseThreads = 1024;

// block-wide exclusive scan of one value per thread; returns the exclusive prefix and, through
// `total`, the block sum. `ws` is a 32-entry scratch.
template <class V>
__device__ __forceinline__ V block_excl_scan(V x, V* ws, V& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  V incl = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const V y = __shfl_up_sync(WHP_FULL, incl, d);
    if (lane >= d) incl += y;
  }
  __syncthreads();  // ws may still be read from a previous call
  if (lane == 31) ws[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    const V v = ws[lane];
    V wi = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const V y = __shfl_up_sync(WHP_FULL, wi, d);
      if (lane >= d) wi += y;
    }
    ws[lane] = wi - v;
    if (lane == 31) ws[32] = wi;
  }
  __syncthreads();
  total = ws[32];
  return ws[warp] + incl - x;
}

// Segment table of the boundary search (phase C below): the plan is cut into n_seg segments of
// seg_len >= C positions; a batch spans at most C positions, so the first batch start at or after
// a segment's first position is one of its first C positions.
constexpr int kMaxSegEntries = 8192;

// SMEM: pre / nxt / mark live in shared memory (and pre, nxt are copied out for the later
// kernels); otherwise they are the global tables themselves (mark = B.bop before it is ranked).
template <bool SMEM>
__global__ void __launch_bounds__(kBaseThreads)
whp_swaps_base_kernel(const whp_tables T, const int32_t* __restrict__ base_perm,
                      const whp_base_tables B, int32_t seg_len, int32_t n_seg) {
  extern __shared__ __align__(16) uint8_t dyn[];
  __shared__ int32_t s_scan32[33];
  dep_trigger();
  const int tid = threadIdx.x;
  const int32_t n = T.n_orders, C = T.C;
  const int32_t n4 = (n + 4) & ~3;  // >= n + 1, a multiple of four (16-byte rows)
  int32_t* pre = SMEM ? reinterpret_cast<int32_t*>(dyn) : B.pre;
  int32_t* nxt = SMEM ? reinterpret_cast<int32_t*>(dyn) + n4 : B.nxt;
  int32_t* mark = SMEM ? reinterpret_cast<int32_t*>(dyn) + 2 * n4 : B.bop;
  int32_t* seg_exit = reinterpret_cast<int32_t*>(dyn) + (SMEM ? 3 * n4 : 0);  // [n_seg][C]
  int32_t* seg_entry = seg_exit + (n_seg > 0 ? n_seg * C : 0);                // [n_seg]

  // ---- A: order record of every position; exclusive prefix of the item counts (four
  // consecutive positions per thread: the dependent global loads of a round overlap)
  const bool vec = (reinterpret_cast<uintptr_t>(base_perm) & 15u) == 0;
  int32_t carry = 0;
  for (int32_t p0 = 0; p0 < n; p0 += 4 * kBaseThreads) {
    const int32_t pb = p0 + 4 * tid;
    const bool full = pb + 3 < n;
    uint32_t orec[4] = {0u, 0u, 0u, 0u};
    if (full && vec) {
      const int4 o = __ldg(reinterpret_cast<const int4*>(base_perm + pb));
      orec[0] = __ldg(T.order_rec + o.x); orec[1] = __ldg(T.order_rec + o.y);
      orec[2] = __ldg(T.order_rec + o.z); orec[3] = __ldg(T.order_rec + o.w);
    } else {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (pb + k < n) orec[k] = __ldg(T.order_rec + __ldg(base_perm + pb + k));
    }
    int32_t qs[4], sum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) { qs[k] = sum; sum += (int32_t)(orec[k] & WHP_Q_MASK); }
    int32_t tot;
    const int32_t ex = carry + block_excl_scan<int32_t>(sum, s_scan32, tot);
    if (full) {
      const int4 pv = make_int4(ex + qs[0], ex + qs[1], ex + qs[2], ex + qs[3]);
      *reinterpret_cast<uint4*>(B.orec + pb) = make_uint4(orec[0], orec[1], orec[2], orec[3]);
      *reinterpret_cast<int4*>(B.pre + pb) = pv;
      if (SMEM) *reinterpret_cast<int4*>(pre + pb) = pv;
    } else {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (pb + k < n) {
          B.orec[pb + k] = orec[k];
          B.pre[pb + k] = ex + qs[k];
          if (SMEM) pre[pb + k] = ex + qs[k];
        }
    }
    carry += tot;
  }
  if (tid == 0) { pre[n] = carry; if (SMEM) B.pre[n] = carry; }
  __syncthreads();

  // ---- B: nxt[p] = where the batch that opens at p ends: the largest e <= min(n, p + C) with
  // pre[e] <= pre[p] + C (q <= C, so e >= p + 1): a binary search; nxt is monotone, so the search
  // of a thread's later positions starts at its predecessor's answer. (A linear advance from
  // there is one step on average but its longest lane holds up the warp.)
  for (int32_t p0 = 0; p0 < n; p0 += 4 * kBaseThreads) {
    const int32_t pb = p0 + 4 * tid;
    if (pb >= n) break;
    int32_t nx[4] = {0, 0, 0, 0};
    int32_t lo = pb + 1;
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (pb + k < n) {
        const int32_t lim = pre[pb + k] + C;
        lo = max(lo, pb + k + 1);
        int32_t hi = min(n, pb + k + C);
        while (lo < hi) {
          const int32_t mid = (lo + hi + 1) >> 1;
          if (pre[mid] <= lim) lo = mid; else hi = mid - 1;
        }
        nx[k] = lo;
      }
    if (pb + 3 < n) {
      const int4 v = make_int4(nx[0], nx[1], nx[2], nx[3]);
      *reinterpret_cast<int4*>(B.nxt + pb) = v;
      if (SMEM) *reinterpret_cast<int4*>(nxt + pb) = v;
      *reinterpret_cast<int4*>(mark + pb) = make_int4(0, 0, 0, 0);
    } else {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (pb + k < n) {
          B.nxt[pb + k] = nx[k];
          if (SMEM) nxt[pb + k] = nx[k];
          mark[pb + k] = 0;
        }
    }
  }
  __syncthreads();

  // ---- C: the base boundaries = the positions reachable from 0 along nxt.
  if (n_seg > 0) {
    // (1) for every segment s and every one of its first C positions: where a chain that passes
    //     through that position enters the next segment
    for (int32_t u = tid; u < n_seg * C; u += kBaseThreads) {
      const int32_t s = u / C;
      int32_t p = s * seg_len + (u - s * C);
      const int32_t lim = min((s + 1) * seg_len, n);
      while (p < lim) p = nxt[p];
      seg_exit[u] = p;
    }
    __syncthreads();
    // (2) one thread composes the segments: the first boundary of each
    if (tid == 0) {
      int32_t E = 0;
      for (int32_t s = 0; s < n_seg; ++s) {
        seg_entry[s] = E;
        if (E < n) E = seg_exit[s * C + (E - s * seg_len)];
      }
    }
    __syncthreads();
    // (3) one thread per segment marks its boundaries
    for (int32_t s = tid; s < n_seg; s += kBaseThreads) {
      const int32_t lim = min((s + 1) * seg_len, n);
      for (int32_t p = seg_entry[s]; p < lim; p = nxt[p]) mark[p] = 1;
    }
  } else if (tid == 0) {  // a table too large for shared memory: one thread chases the boundaries
    for (int32_t p = 0; p < n; p = nxt[p]) mark[p] = 1;
  }
  __syncthreads();
  // ---- D: a block scan ranks the marks (bstart[b], bop[p])
  int32_t carry_b = 0;
  for (int32_t p0 = 0; p0 < n; p0 += 4 * kBaseThreads) {  // four positions per thread
    const int32_t pb = p0 + 4 * tid;
    int32_t mk[4], before[4], sum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      mk[k] = (pb + k < n) ? mark[pb + k] : 0;
      before[k] = sum;
      sum += mk[k];
    }
    int32_t tot;
    const int32_t ex = carry_b + block_excl_scan<int32_t>(sum, s_scan32, tot);
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (pb + k < n) {
        const int32_t rank = ex + before[k];
        if (mk[k]) B.bstart[rank] = pb + k;
        B.bop[pb + k] = rank + mk[k] - 1;
      }
    carry_b += tot;
  }
  if (tid == 0) { B.bstart[carry_b] = n; B.totals[1] = carry_b; }
}

// Second half of the base pass, after whp_swaps_prep_kernel has scored the base batches
// (dist_at / cls_at at their start positions); blocks 0 .. KW of whp_swaps_tail_kernel.
// Block w < KW: the class-count prefix rpre[b][k] of the 32 classes of word w, over chunks of 32
// batches: lane j of the chunk's warp gets the ballot of class j over the chunk's batches, a
// two-level running sum (chunks of a warp, then warps) gives the chunk's offset, and row b of the
// chunk is offset + popc(ballot below b) — one coalesced row store per batch, no read-modify-write
// of global memory. Block KW: the prefix of the batch lengths (bdist[nb] = D_base).
// s_tab: [2 * 32 * chunk_cap + 1024] words of shared memory.
constexpr int kBase2ChunkCap = 256;  // chunks (of 32 batches) the shared-memory path takes

__device__ __forceinline__ void base2_role(const whp_tables& T, const whp_base_tables& B,
                                           int32_t* s_tab, int32_t chunk_cap) {
  __shared__ int64_t s_scan64[33];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int32_t nb = (int32_t)B.totals[1];
  const int KW = (T.K + 31) >> 5;
  if ((int)blockIdx.x == KW) {
    int64_t carry64 = 0;
    for (int32_t b0 = 0; b0 <= nb; b0 += kBaseThreads) {
      const int32_t b = b0 + tid;
      const int64_t x = (b < nb) ? B.dist_at[B.bstart[b]] : 0;
      int64_t tot;
      const int64_t ex = block_excl_scan<int64_t>(x, s_scan64, tot);
      if (b <= nb) B.bdist[b] = carry64 + ex;
      carry64 += tot;
    }
    if (tid == 0) B.totals[0] = carry64;
    return;
  }
  const int w = blockIdx.x;
  const bool mine = 32 * w + lane < T.K;
  const int32_t nchunks = (nb + 31) >> 5;
  int32_t* __restrict__ row = B.rpre + 32 * w + lane;
  if (nchunks <= chunk_cap) {
    int32_t* s_off = s_tab;                   // [chunk][class]: visits in the warp's chunks before
    int32_t* s_msk = s_tab + 32 * chunk_cap;  // [chunk][class]: ballot of the class over the chunk
    int32_t* s_seg = s_tab + 64 * chunk_cap;  // [warp][class]: visits in the warp's chunks
    const int32_t per = (nchunks + 31) >> 5;  // chunks per warp
    const int32_t c_lo = min(warp * per, nchunks), c_hi = min(c_lo + per, nchunks);
    int32_t run = 0;
    for (int32_t c = c_lo; c < c_hi; ++c) {
      const int32_t b = 32 * c + lane;
      const uint32_t word = (b < nb) ? B.cls_at[(int64_t)B.bstart[b] * 8 + w] : 0u;
      uint32_t m = 0;
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        const uint32_t bal = __ballot_sync(WHP_FULL, (word >> j) & 1u);
        if (lane == j) m = bal;
      }
      s_off[32 * c + lane] = run;
      s_msk[32 * c + lane] = (int32_t)m;
      run += __popc(m);
    }
    s_seg[32 * warp + lane] = run;
    __syncthreads();
    int32_t off = 0;
    for (int s2 = 0; s2 < warp; ++s2) off += s_seg[32 * s2 + lane];
    if (warp == kBaseThreads / 32 - 1 && mine) {  // the last warp's offset + its own = the total
      B.resp[32 * w + lane] = off + run;
      row[(int64_t)nb * T.K] = off + run;
    }
    for (int32_t c = c_lo; c < c_hi; ++c) {
      const int32_t base = off + s_off[32 * c + lane];
      const uint32_t m = (uint32_t)s_msk[32 * c + lane];
      const int nbb = min(32, nb - 32 * c);
      if (mine)
        for (int bb = 0; bb < nbb; ++bb)
          row[(int64_t)(32 * c + bb) * T.K] = base + __popc(m & ((1u << bb) - 1u));
    }
    return;
  }
  // more batches than the shared-memory tables take: the chunk totals are parked in the rows
  // themselves (row 32c+1, rewritten below) and one warp runs over the chunks
  for (int32_t c = warp; c < nchunks; c += kBaseThreads / 32) {
    const int32_t b = 32 * c + lane;
    const uint32_t word = (b < nb) ? B.cls_at[(int64_t)B.bstart[b] * 8 + w] : 0u;
    int32_t tot = 0;
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      const int32_t pc = __popc(__ballot_sync(WHP_FULL, (word >> j) & 1u));
      if (lane == j) tot = pc;
    }
    if (mine) row[(int64_t)(32 * c + 1) * T.K] = tot;
  }
  __syncthreads();
  if (warp == 0 && mine) {
    int32_t run = 0;
    for (int32_t c = 0; c < nchunks; ++c) {
      const int32_t t = row[(int64_t)(32 * c + 1) * T.K];
      row[(int64_t)(32 * c) * T.K] = run;
      run += t;
    }
    if (nchunks == 0) row[0] = 0;
    B.resp[32 * w + lane] = run;
  }
  __syncthreads();
  for (int32_t c = warp; c < nchunks; c += kBaseThreads / 32) {
    const int32_t b = 32 * c + lane;
    const uint32_t word = (b < nb) ? B.cls_at[(int64_t)B.bstart[b] * 8 + w] : 0u;
    int32_t cnt = mine ? row[(int64_t)(32 * c) * T.K] : 0;
    const int nbb = min(32, nb - 32 * c);
    for (int bb = 0; bb < nbb; ++bb) {
      cnt += (int32_t)((__shfl_sync(WHP_FULL, word, bb) >> lane) & 1u);
      if (mine) row[(int64_t)(32 * c + bb + 1) * T.K] = cnt;
    }
  }
}

// ------------------------------------------------------------------------------ region prep
// For every position p of the region [rlo, rhi): the batch that WOULD open at p in the base
// plan, [p, nxt[p]) — its S-shape length dist_at[p] and class mask cls_at[p]. A rescored plan
// differs from the base plan only around the two swapped positions; every other new batch is
// one of these (its end depends on its start alone), so a neighbour looks it up.
constexpr int kPrepWarps = 8;

__global__ void __launch_bounds__(kPrepWarps * 32)
whp_swaps_prep_kernel(const whp_tables T, const whp_base_tables B, int32_t rlo, int32_t rhi) {
  __shared__ warp_sets sets_all[kPrepWarps];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  warp_sets* sets = &sets_all[warp];
  sets->amask[lane] = 0;
  if (lane < 8) sets->cmask[lane] = 0;
  dep_wait();
  dep_trigger();
  __syncwarp();
  // warps 0 .. rows-1: the region positions; the others: the base batches (their starts)
  const int32_t g = blockIdx.x * kPrepWarps + warp;
  int32_t p;
  if (g < rhi - rlo) {
    p = rlo + g;
  } else {
    const int32_t b = g - (rhi - rlo);
    if (b >= (int32_t)B.totals[1]) return;
    p = B.bstart[b];
    if (p >= rlo && p < rhi) return;  // scored as a region position
  }
  swap_seq q{B.pre, B.orec, nullptr, nullptr, 0, 0u, 0u, -1, -1, 0};
  const int64_t dist = score_batch(T, sets, q, p, B.nxt[p]);
  if (lane == 0) B.dist_at[p] = dist;
  if (lane < 8) B.cls_at[(int64_t)p * 8 + lane] = sets->cmask[lane];
}

// ------------------------------------------------------------------------------ chains
// A plan re-batched from position p follows p -> nxt[p] -> nxt[nxt[p]] ... until a start
// coincides with a base batch start F(p) (from there on it IS the base plan). That chain depends
// on p alone, and two next-fit chains take long to meet (tens of batches), so it is summed once
// per region position: dtail[p] = lengths of the chain's batches before F(p), rtail[p][k] = their
// class visits, bF[p] = base batch that starts at F(p) (nb: the chain runs to the end of the plan;
// -1: it leaves the region first). With T(p) = dtail[p] + (D_base - bdist[bF[p]]), any stretch
// s -> t of one chain costs T(s) - T(t).
// Only the chains of the positions a neighbour can ask for are summed: the first new boundary
// after the later swapped position lies at most C positions behind it, so p < chi = window end +
// C + 1 (and once a chain has left the region, so has every later node of it).
constexpr int kChainWarps = 4;  // warps of a block that walk one chain each

template <int BYTES>
__device__ __forceinline__ void stage_async(void* smem_dst, const void* gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(
                   (uint32_t)__cvta_generic_to_shared(smem_dst)),
               "l"(gmem_src), "n"(BYTES)
               : "memory");
}

// One launch after whp_swaps_prep_kernel: blocks 0 .. KW are the second half of the base pass
// (base2_role), the others sum kChainWarps chains each. The two halves are independent.
// STAGED: the hop records of the region sit in shared memory (a chain only moves forward, so a
// block stages the rows from its own first position on); otherwise (a region too long for
// shared memory) they are read from global memory.
template <bool STAGED>
__global__ void __launch_bounds__(kBaseThreads)
whp_swaps_tail_kernel(const whp_tables T, const whp_base_tables B, int32_t rlo, int32_t rhi,
                      int32_t chi, int32_t chunk_cap) {
  // chain blocks: [cls_at: rows x 8][dist_at: rows (int64)][nxt: rows; negative: p is a base
  // batch start][bop: rows + 1]; base2 blocks: see base2_role
  extern __shared__ __align__(16) uint8_t chain_smem[];
  dep_wait();
  const int KW = (T.K + 31) >> 5;
  if ((int)blockIdx.x <= KW) {
    base2_role(T, B, reinterpret_cast<int32_t*>(chain_smem), chunk_cap);
    return;
  }
  const int32_t r0 = rlo + ((int)blockIdx.x - KW - 1) * kChainWarps;  // first position of this block
  const int32_t rows = STAGED ? rhi - r0 : 0;
  uint4* s_cls = reinterpret_cast<uint4*>(chain_smem);
  int64_t* s_dist = reinterpret_cast<int64_t*>(chain_smem + 32 * (size_t)rows);
  int32_t* s_nx = reinterpret_cast<int32_t*>(chain_smem + 40 * (size_t)rows);
  int32_t* s_bop = reinterpret_cast<int32_t*>(chain_smem + 44 * (size_t)rows);  // bop[r0-1 .. rhi)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int32_t n = T.n_orders;
  if (STAGED) {
    // asynchronous copies: every load of the block is in flight before the first one is awaited
    const uint4* cls_src = reinterpret_cast<const uint4*>(B.cls_at + (int64_t)r0 * 8);
    for (int32_t k = threadIdx.x; k < 2 * rows; k += blockDim.x) stage_async<16>(s_cls + k, cls_src + k);
    for (int32_t k = threadIdx.x; k < rows; k += blockDim.x) {
      stage_async<8>(s_dist + k, B.dist_at + r0 + k);
      stage_async<4>(s_nx + k, B.nxt + r0 + k);
    }
    for (int32_t k = threadIdx.x; k <= rows; k += blockDim.x) {
      if (r0 + k > 0) stage_async<4>(s_bop + k, B.bop + r0 - 1 + k);
      else s_bop[k] = -1;
    }
    asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    for (int32_t k = threadIdx.x; k < rows; k += blockDim.x)
      if (s_bop[k + 1] != s_bop[k]) s_nx[k] = -1;  // position r0 + k opens a base batch
    __syncthreads();
  }
  const int32_t p0 = r0 + warp;
  if (warp >= kChainWarps || p0 >= chi) return;
  int64_t D = 0;
  int32_t r[8];
#pragma unroll
  for (int w = 0; w < 8; ++w) r[w] = 0;
  int32_t p = p0, bF;
  for (;;) {
    if (p >= n) { bF = (int32_t)B.totals[1]; break; }
    if (p >= rhi) { bF = -1; break; }
    int32_t nx;
    uint4 c0, c1;
    if (STAGED) {
      nx = s_nx[p - r0];
      if (nx < 0) { bF = B.bop[p]; break; }
      D += s_dist[p - r0];
      c0 = s_cls[2 * (p - r0)];
      c1 = s_cls[2 * (p - r0) + 1];
    } else {
      if (p == 0 || B.bop[p] != B.bop[p - 1]) { bF = B.bop[p]; break; }
      nx = B.nxt[p];
      D += B.dist_at[p];
      c0 = reinterpret_cast<const uint4*>(B.cls_at + (int64_t)p * 8)[0];
      c1 = reinterpret_cast<const uint4*>(B.cls_at + (int64_t)p * 8)[1];
    }
    r[0] += (int32_t)((c0.x >> lane) & 1u); r[1] += (int32_t)((c0.y >> lane) & 1u);
    r[2] += (int32_t)((c0.z >> lane) & 1u); r[3] += (int32_t)((c0.w >> lane) & 1u);
    r[4] += (int32_t)((c1.x >> lane) & 1u); r[5] += (int32_t)((c1.y >> lane) & 1u);
    r[6] += (int32_t)((c1.z >> lane) & 1u); r[7] += (int32_t)((c1.w >> lane) & 1u);
    p = nx;
  }
  if (lane == 0) { B.dtail[p0] = D; B.bF[p0] = bF; }
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    const int k = 32 * w + lane;
    if (k < T.K) B.rtail[(int64_t)(p0 - rlo) * T.K + k] = r[w];
  }
}

// ------------------------------------------------------------------------------ neighbours
constexpr int kSwapWarps = 8;
constexpr int kStage = 1024;  // positions of pre / orec staged per block

template <bool STATS>  // STATS: also count the batches / picks scored from their picks
__global__ void __launch_bounds__(kSwapWarps * 32)
whp_swaps_kernel(const whp_tables T, const whp_base_tables B, int32_t win_start, int32_t W,
                 int32_t rlo, int32_t rhi, int32_t chi, int64_t n_nb,
                 int64_t* __restrict__ d_dist, double* __restrict__ d_obj,
                 unsigned long long* __restrict__ stats) {
  __shared__ warp_sets sets_all[kSwapWarps];
  __shared__ int32_t s_pre[kStage + 1];
  __shared__ uint32_t s_orec[kStage];
  __shared__ int32_t s_nxt[kStage];
  uint32_t n_scored = 0, n_scored_picks = 0;  // stats: batches / picks scored from their picks
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  warp_sets* sets = &sets_all[warp];
  sets->amask[lane] = 0;
  if (lane < 8) sets->cmask[lane] = 0;
  const int32_t n = T.n_orders;
  const int32_t nb = (int32_t)B.totals[1];
  // stage the tables from the start of the batch before the window's first batch
  int32_t lo;
  {
    const int32_t bw = __ldg(B.bop + win_start);
    lo = __ldg(B.bstart + (bw > 0 ? bw - 1 : 0));
  }
  // (what a neighbour reads lies between that start and a cart or two past the window; anything
  // further goes through the accessors' global-memory path)
  const int32_t cnt = min(min(kStage, n - lo), win_start + W + 3 * T.C + 32 - lo);
  for (int k = threadIdx.x; k <= cnt; k += blockDim.x) s_pre[k] = __ldg(B.pre + lo + k);
  for (int k = threadIdx.x; k < cnt; k += blockDim.x) s_orec[k] = __ldg(B.orec + lo + k);
  for (int k = threadIdx.x; k < cnt; k += blockDim.x) s_nxt[k] = __ldg(B.nxt + lo + k);
  __syncthreads();
  const int64_t D_base = B.totals[0];
  auto nxt_at = [&](int32_t p) -> int32_t {
    const uint32_t k = (uint32_t)(p - lo);
    return k < (uint32_t)cnt ? s_nxt[k] : __ldg(B.nxt + p);
  };

  for (int64_t nn = (int64_t)blockIdx.x * kSwapWarps + warp; nn < n_nb;
       nn += (int64_t)gridDim.x * kSwapWarps) {
    // neighbour index -> (i', j'), row i' starts at i'(2W-i'-1)/2
    // (an estimate of the row by a square root, made exact by the two integer loops; windows
    // below 32,768 positions — W^2 < 2^30 — take 32-bit arithmetic and a float estimate)
    int32_t pi, pj;
    if (W < 32768) {
      const int32_t n32 = (int32_t)nn, w2 = 2 * W;
      const float wm = (float)(w2 - 1);
      int32_t i = (int32_t)((wm - sqrtf(fmaxf(wm * wm - 8.0f * (float)n32, 0.0f))) * 0.5f);
      i = max(0, min(i, W - 2));
      while (i > 0 && i * (w2 - i - 1) / 2 > n32) --i;
      while ((i + 1) * (w2 - i - 2) / 2 <= n32) ++i;
      pi = win_start + i;
      pj = pi + 1 + (n32 - i * (w2 - i - 1) / 2);
    } else {
      const double wm = 2.0 * W - 1.0;
      int64_t i = (int64_t)floor((wm - sqrt(wm * wm - 8.0 * (double)nn)) * 0.5);
      i = max((int64_t)0, min(i, (int64_t)W - 2));
      while (i > 0 && i * (2 * (int64_t)W - i - 1) / 2 > nn) --i;
      while ((i + 1) * (2 * (int64_t)W - i - 2) / 2 <= nn) ++i;
      const int64_t j = i + 1 + (nn - i * (2 * (int64_t)W - i - 1) / 2);
      pi = win_start + (int32_t)i;
      pj = win_start + (int32_t)j;
    }
    const int32_t bi = __ldg(B.bop + pi), bj = __ldg(B.bop + pj);
    swap_seq q{B.pre, B.orec, s_pre, s_orec, lo, (uint32_t)(cnt + 1), (uint32_t)cnt, pi, pj, 0};
    const int32_t qi = (int32_t)(q.orec_at(pj) & WHP_Q_MASK);  // orec_at swaps: this is q(pi)
    const int32_t qj = (int32_t)(q.orec_at(pi) & WHP_Q_MASK);
    q.delta = qj - qi;
    // a smaller order arriving at the opening position of a cart may slip into the cart before
    const bool slip = q.delta < 0 && bi > 0 && pi == __ldg(B.bstart + bi);
    if (bi == bj && !slip) {  // both orders stay in the same cart: nothing changes
      int32_t rb[8];
#pragma unroll
      for (int w = 0; w < 8; ++w) rb[w] = (32 * w + lane < T.K) ? __ldg(B.resp + 32 * w + lane) : 0;
      const double phi_base = penalty_regs(T, rb);
      if (lane == 0) {
        if (d_dist) d_dist[nn] = D_base;
        if (d_obj) d_obj[nn] = __dadd_rn((double)D_base, phi_base);
      }
      continue;
    }

    int64_t D = D_base;
    int32_t r[8];
#pragma unroll
    for (int w = 0; w < 8; ++w) r[w] = 0;
    auto add_classes = [&]() {  // new batch: + its classes, then clear the mask
      __syncwarp();
#pragma unroll
      for (int w = 0; w < 8; ++w) r[w] += (int32_t)((sets->cmask[w] >> lane) & 1u);
      __syncwarp();
      if (lane < 8) sets->cmask[lane] = 0;
      __syncwarp();
    };
    auto remove_base = [&](int32_t b_from, int32_t b_to) {  // base batches [b_from, b_to)
      D -= B.bdist[b_to] - B.bdist[b_from];
#pragma unroll
      for (int w = 0; w < 8; ++w) {
        const int k = 32 * w + lane;
        if (k < T.K)
          r[w] -= __ldg(B.rpre + (int64_t)b_to * T.K + k) - __ldg(B.rpre + (int64_t)b_from * T.K + k);
      }
    };
    if (q.delta == 0) {
      // boundaries stay: rescore the two carts that exchange an order
      remove_base(bi, bi + 1);
      remove_base(bj, bj + 1);
      D += score_batch(T, sets, q, __ldg(B.bstart + bi), __ldg(B.bstart + bi + 1));
      add_classes();
      D += score_batch(T, sets, q, __ldg(B.bstart + bj), __ldg(B.bstart + bj + 1));
      add_classes();
      if (STATS) {
        n_scored += 2;
        n_scored_picks += (uint32_t)(q.pre_at(__ldg(B.bstart + bi + 1)) - q.pre_at(__ldg(B.bstart + bi)) +
                                     q.pre_at(__ldg(B.bstart + bj + 1)) - q.pre_at(__ldg(B.bstart + bj)));
      }
    } else {
      const int32_t b0 = slip ? bi - 1 : bi;
      int32_t p = __ldg(B.bstart + b0);
      int32_t b_end;
      for (;;) {
        // (1) past pj the rest of the rewalk is the chain of p, summed once per position
        if (p > pj && p >= rlo && p < chi) {
          const int32_t bf = __ldg(B.bF + p);
          if (bf >= 0) {
            D += __ldg(B.dtail + p);
#pragma unroll
            for (int w = 0; w < 8; ++w) {
              const int k = 32 * w + lane;
              if (k < T.K) r[w] += __ldg(B.rtail + (int64_t)(p - rlo) * T.K + k);
            }
            b_end = bf;
            break;
          }
        }
        // (2) between pi and pj the prefix is shifted uniformly: batches that end before pj
        // are the chain of p as well — hop to its last node t before pj, add T(p) - T(t)
        if (p > pi && p < pj && p >= rlo && pj < rhi) {
          int32_t t = p;
          for (int32_t nx = nxt_at(t); nx < pj; nx = nxt_at(t)) t = nx;
          if (t != p) {
            const int32_t bfp = __ldg(B.bF + p), bft = __ldg(B.bF + t);
            if (bfp >= 0 && bft >= 0) {
              D += (__ldg(B.dtail + p) - __ldg(B.dtail + t)) + (B.bdist[bft] - B.bdist[bfp]);
#pragma unroll
              for (int w = 0; w < 8; ++w) {
                const int k = 32 * w + lane;
                if (k < T.K) {
                  r[w] += __ldg(B.rtail + (int64_t)(p - rlo) * T.K + k) -
                          __ldg(B.rtail + (int64_t)(t - rlo) * T.K + k);
                  if (bft != bfp)
                    r[w] += __ldg(B.rpre + (int64_t)bft * T.K + k) - __ldg(B.rpre + (int64_t)bfp * T.K + k);
                }
              }
              p = t;
            }
          }
        }
        // A batch that holds neither swapped position and ends where the base criterion ends
        int32_t e;
        bool table;
        if (p > pj) {
          e = __ldg(B.nxt + p);
          table = true;
        } else {
          e = batch_end(q, p, n, T.C);
          table = (p > pi || e <= pi) && e <= pj && __ldg(B.nxt + p) == e;
        }
        if (table && p >= rlo && p < rhi) {
          D += __ldg(B.dist_at + p);
          const uint4 c0 = __ldg(reinterpret_cast<const uint4*>(B.cls_at + (int64_t)p * 8));
          const uint4 c1 = __ldg(reinterpret_cast<const uint4*>(B.cls_at + (int64_t)p * 8) + 1);
          r[0] += (int32_t)((c0.x >> lane) & 1u); r[1] += (int32_t)((c0.y >> lane) & 1u);
          r[2] += (int32_t)((c0.z >> lane) & 1u); r[3] += (int32_t)((c0.w >> lane) & 1u);
          r[4] += (int32_t)((c1.x >> lane) & 1u); r[5] += (int32_t)((c1.y >> lane) & 1u);
          r[6] += (int32_t)((c1.z >> lane) & 1u); r[7] += (int32_t)((c1.w >> lane) & 1u);
        } else {
          D += score_batch(T, sets, q, p, e);
          add_classes();
          if (STATS) { n_scored += 1; n_scored_picks += (uint32_t)(q.pre_at(e) - q.pre_at(p)); }
        }
        p = e;
        if (p >= n) { b_end = nb; break; }
        if (p > pj && __ldg(B.bop + p) != __ldg(B.bop + p - 1)) { b_end = __ldg(B.bop + p); break; }
      }
      remove_base(b0, b_end);
    }
#pragma unroll
    for (int w = 0; w < 8; ++w) {
      const int k = 32 * w + lane;
      if (k < T.K) r[w] += __ldg(B.resp + k);
    }
    const double phi = penalty_regs(T, r);
    if (lane == 0) {
      if (d_dist) d_dist[nn] = D;
      if (d_obj) d_obj[nn] = __dadd_rn((double)D, phi);
    }
  }
  if (STATS && lane == 0) {
    atomicAdd(stats, (unsigned long long)n_scored);
    atomicAdd(stats + 1, (unsigned long long)n_scored_picks);
  }
}

// ------------------------------------------------------------------------------ NEXT-4: moves
// Insertion neighbourhood (reading N4): one warp per move (i' -> j'). The plan is re-batched
// from the cart of the first changed position m = min(pi, pj) (one cart earlier when m opens
// its cart: a different order there may slip back) until, after M = max(pi, pj), a new boundary
// coincides with a base boundary. The orders between pi and pj only shift by one position, so a
// new batch that lies between them and ends where the base criterion ends it is the tabulated
// batch of its (shifted) base start; after M the rest is one chain look-up, as for swaps.
template <bool STATS>
__global__ void __launch_bounds__(kSwapWarps * 32)
whp_moves_kernel(const whp_tables T, const whp_base_tables B, int32_t win_start, int32_t W,
                 int32_t rlo, int32_t rhi, int32_t chi, int64_t n_nb,
                 int64_t* __restrict__ d_dist, double* __restrict__ d_obj,
                 unsigned long long* __restrict__ stats) {
  __shared__ warp_sets sets_all[kSwapWarps];
  __shared__ int32_t s_pre[kStage + 1];
  __shared__ uint32_t s_orec[kStage];
  uint32_t n_scored = 0, n_scored_picks = 0;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  warp_sets* sets = &sets_all[warp];
  sets->amask[lane] = 0;
  if (lane < 8) sets->cmask[lane] = 0;
  const int32_t n = T.n_orders;
  const int32_t nb = (int32_t)B.totals[1];
  int32_t lo;
  {
    const int32_t bw = __ldg(B.bop + win_start);
    lo = __ldg(B.bstart + (bw > 0 ? bw - 1 : 0));
  }
  const int32_t cnt = min(kStage, n - lo);
  for (int k = threadIdx.x; k <= cnt; k += blockDim.x) s_pre[k] = __ldg(B.pre + lo + k);
  for (int k = threadIdx.x; k < cnt; k += blockDim.x) s_orec[k] = __ldg(B.orec + lo + k);
  __syncthreads();
  const int64_t D_base = B.totals[0];
  for (int64_t nn = (int64_t)blockIdx.x * kSwapWarps + warp; nn < n_nb;
       nn += (int64_t)gridDim.x * kSwapWarps) {
    // (32-bit division when the neighbourhood has fewer than 2^31 moves)
    const int32_t i = n_nb <= 0x7fffffff ? (int32_t)((uint32_t)nn / (uint32_t)(W - 1))
                                         : (int32_t)(nn / (W - 1));
    const int32_t jr = (int32_t)(nn - (int64_t)i * (W - 1));
    const int32_t j = jr < i ? jr : jr + 1;
    const int32_t pi = win_start + i, pj = win_start + j;
    const int32_t m = min(pi, pj), M = max(pi, pj);
    move_seq q{B.pre, B.orec, s_pre, s_orec, lo, (uint32_t)(cnt + 1), (uint32_t)cnt, pi, pj, 0};
    q.qi = q.pre_base(pi + 1) - q.pre_base(pi);
    int32_t b0 = __ldg(B.bop + m);
    if (b0 > 0 && m == __ldg(B.bstart + b0)) b0 -= 1;  // a different order opens the cart: may slip
    int32_t p = __ldg(B.bstart + b0);
    int64_t D = D_base;
    int32_t r[8];
#pragma unroll
    for (int w = 0; w < 8; ++w) r[w] = 0;
    int32_t b_end;
    for (;;) {
      if (p > M && p >= rlo && p < chi) {  // the rest is the chain of p
        const int32_t bf = __ldg(B.bF + p);
        if (bf >= 0) {
          D += __ldg(B.dtail + p);
#pragma unroll
          for (int w = 0; w < 8; ++w) {
            const int k = 32 * w + lane;
            if (k < T.K) r[w] += __ldg(B.rtail + (int64_t)(p - rlo) * T.K + k);
          }
          b_end = bf;
          break;
        }
      }
      const int32_t e = batch_end(q, p, n, T.C);
      // base start of the batch if it is a run of base orders in base order: before m, after
      // M, or between pi and pj without the re-inserted order (positions shifted by one)
      int32_t bp = -1;
      if (e <= m || p > M) bp = p;
      else if (pi < pj && p >= pi && e <= pj) bp = p + 1;
      else if (pj < pi && p > pj && e <= pi + 1) bp = p - 1;
      if (bp >= rlo && bp < rhi && __ldg(B.nxt + bp) == bp + (e - p)) {
        D += __ldg(B.dist_at + bp);
        const uint4 c0 = __ldg(reinterpret_cast<const uint4*>(B.cls_at + (int64_t)bp * 8));
        const uint4 c1 = __ldg(reinterpret_cast<const uint4*>(B.cls_at + (int64_t)bp * 8) + 1);
        r[0] += (int32_t)((c0.x >> lane) & 1u); r[1] += (int32_t)((c0.y >> lane) & 1u);
        r[2] += (int32_t)((c0.z >> lane) & 1u); r[3] += (int32_t)((c0.w >> lane) & 1u);
        r[4] += (int32_t)((c1.x >> lane) & 1u); r[5] += (int32_t)((c1.y >> lane) & 1u);
        r[6] += (int32_t)((c1.z >> lane) & 1u); r[7] += (int32_t)((c1.w >> lane) & 1u);
      } else {
        D += score_batch(T, sets, q, p, e);
        if (STATS) { n_scored += 1; n_scored_picks += (uint32_t)(q.pre_at(e) - q.pre_at(p)); }
        __syncwarp();
#pragma unroll
        for (int w = 0; w < 8; ++w) r[w] += (int32_t)((sets->cmask[w] >> lane) & 1u);
        __syncwarp();
        if (lane < 8) sets->cmask[lane] = 0;
        __syncwarp();
      }
      p = e;
      if (p >= n) { b_end = nb; break; }
      if (p > M && __ldg(B.bop + p) != __ldg(B.bop + p - 1)) { b_end = __ldg(B.bop + p); break; }
    }
    D -= B.bdist[b_end] - B.bdist[b0];
#pragma unroll
    for (int w = 0; w < 8; ++w) {
      const int k = 32 * w + lane;
      if (k < T.K)
        r[w] += __ldg(B.resp + k) - (__ldg(B.rpre + (int64_t)b_end * T.K + k) -
                                     __ldg(B.rpre + (int64_t)b0 * T.K + k));
    }
    const double phi = penalty_regs(T, r);
    if (lane == 0) {
      if (d_dist) d_dist[nn] = D;
      if (d_obj) d_obj[nn] = __dadd_rn((double)D, phi);
    }
  }
  if (STATS && lane == 0) {
    atomicAdd(stats, (unsigned long long)n_scored);
    atomicAdd(stats + 1, (unsigned long long)n_scored_picks);
  }
}

// apply move *d_idx (as written by whp_argmin over a whp_eval_moves result) to the plan
__global__ void whp_apply_move_kernel(int32_t* __restrict__ base_perm, int32_t win_start, int32_t W,
                                      const int64_t* __restrict__ d_idx) {
  const int64_t nn = *d_idx;
  if (nn < 0 || nn >= (int64_t)W * (W - 1)) return;
  const int32_t i = (int32_t)(nn / (W - 1));
  const int32_t jr = (int32_t)(nn - (int64_t)i * (W - 1));
  const int32_t j = jr < i ? jr : jr + 1;
  const int32_t from = win_start + i, to = win_start + j;
  const int32_t moved = base_perm[from];
  if (from < to) for (int32_t q = from; q < to; ++q) base_perm[q] = base_perm[q + 1];
  else for (int32_t q = from; q > to; --q) base_perm[q] = base_perm[q - 1];
  base_perm[to] = moved;
}

}  // namespace

// base pass + region tables + chain sums of one window (shared by the swap and the move
// neighbourhoods)
static cudaError_t launch_window_tables(whp_ctx* c, const whp_tables& T, const int32_t* d_base_perm,
                                        int32_t win_start, int32_t win_len, int32_t* rlo_out,
                                        int32_t* rhi_out, int32_t* chi_out, cudaStream_t st) {
  // boundary search of the base pass: segments of seg_len >= C positions, about 1024 / C of them
  // (one thread per (segment, entry position) pair); without a table (n_seg = 0) one thread chases
  const int64_t n64 = c->n_orders, C64 = c->C;
  int64_t seg_len = (n64 * C64 + kBaseThreads - 1) / kBaseThreads;
  if (seg_len < C64) seg_len = C64;
  if (seg_len > n64) seg_len = n64;  // C > n: one segment
  int64_t n_seg = (n64 + seg_len - 1) / seg_len;
  if (n_seg * C64 > kMaxSegEntries) n_seg = 0;
  const size_t seg_bytes = 4 * (size_t)(n_seg * C64 + n_seg);
  // shared-memory tables of the base pass: pre, nxt and the boundary marks, when they fit
  const size_t n4 = ((size_t)c->n_orders + 4) & ~(size_t)3;
  const size_t need = 12 * n4 + seg_bytes;
  const bool smem_tables = need + 12 * 1024 <= (size_t)c->smem_optin;
  // the attribute is per function and process-wide: always the same value (the most any call
  // asks for), so contexts used from different host threads cannot undercut each other
  cudaError_t e = cudaFuncSetAttribute(whp_swaps_base_kernel<true>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       c->smem_optin - 12 * 1024);
  if (e != cudaSuccess) return e;
  if (smem_tables)
    whp_swaps_base_kernel<true><<<1, kBaseThreads, need, st>>>(T, d_base_perm, c->base,
                                                               (int32_t)seg_len, (int32_t)n_seg);
  else
    whp_swaps_base_kernel<false><<<1, kBaseThreads, seg_bytes, st>>>(T, d_base_perm, c->base,
                                                                     (int32_t)seg_len, (int32_t)n_seg);
  c->launches += 1;
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  // region of tabulated hypothetical batches: from two cart lengths before the window (the
  // rewalk may start one batch early) to a margin after it (until the boundaries resynchronise;
  // beyond the margin a neighbour scores its batches from their picks)
  // (two next-fit chains need a median of ~150 positions to meet at paper scale, but the tail is
  // long: with 512 positions one window in five still had chains that left the region, and every
  // neighbour that lands on such a chain then scores tens of batches from their picks)
  int64_t margin = 64ll * c->C > 2048 ? 64ll * c->C : 2048;
  if (c->dbg_swap_margin >= 0) margin = c->dbg_swap_margin;  // WHP_DEBUG_SWAP_MARGIN: tests force the fallbacks
  const int32_t rlo = (int32_t)((int64_t)win_start - 2ll * c->C > 0 ? (int64_t)win_start - 2ll * c->C : 0);
  const int32_t rhi = (int32_t)((int64_t)win_start + win_len + margin < c->n_orders
                                    ? (int64_t)win_start + win_len + margin : c->n_orders);
  // hypothetical batches of the region and the base batches themselves
  int64_t nb_max = 2ll * c->n_items / ((int64_t)c->C + 1) + 1;
  if (nb_max > c->n_orders) nb_max = c->n_orders;
  if ((e = launch_dependent(whp_swaps_prep_kernel,
                            (unsigned)((rhi - rlo + nb_max + kPrepWarps - 1) / kPrepWarps),
                            kPrepWarps * 32, 0, st, T, c->base, rlo, rhi)) != cudaSuccess) return e;
  c->launches += 1;
  // second half of the base pass and the chain sums of the positions a neighbour can ask for,
  // in one launch (rtail grows with the window)
  const int32_t chi = (int32_t)((int64_t)win_start + win_len + c->C + 1 < rhi
                                    ? (int64_t)win_start + win_len + c->C + 1 : rhi);
  const int64_t rows = chi - rlo;
  if (c->rtail_rows < rows) {
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return e;
    cudaFree(c->base.rtail);
    c->base.rtail = nullptr;
    c->rtail_rows = 0;
    if ((e = cudaMalloc(&c->base.rtail, 4 * (size_t)rows * (size_t)c->K)) != cudaSuccess) return e;
    c->rtail_rows = rows;
  }
  int64_t chunk_cap = nb_max / 32 + 1;
  if (chunk_cap > kBase2ChunkCap) chunk_cap = kBase2ChunkCap;
  const size_t base2_smem = 4 * (64 * (size_t)chunk_cap + 1024);
  const size_t chain_smem = 48 * (size_t)(rhi - rlo) + 16;
  const unsigned tail_blocks = (unsigned)((c->K + 31) / 32 + 1 + (rows + kChainWarps - 1) / kChainWarps);
  if ((e = cudaFuncSetAttribute(whp_swaps_tail_kernel<true>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize,
                                c->smem_optin - 2048)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(whp_swaps_tail_kernel<false>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize,
                                c->smem_optin - 2048)) != cudaSuccess) return e;
  if (chain_smem + 2048 <= (size_t)c->smem_optin)
    e = launch_dependent(whp_swaps_tail_kernel<true>, tail_blocks, kBaseThreads,
                         chain_smem > base2_smem ? chain_smem : base2_smem, st, T, c->base, rlo,
                         rhi, chi, (int32_t)chunk_cap);
  else
    e = launch_dependent(whp_swaps_tail_kernel<false>, tail_blocks, kBaseThreads, base2_smem, st, T,
                         c->base, rlo, rhi, chi, (int32_t)chunk_cap);
  if (e != cudaSuccess) return e;
  c->launches += 1;
  *rlo_out = rlo;
  *rhi_out = rhi;
  *chi_out = chi;
  return cudaSuccess;
}

cudaError_t whp_launch_swaps(whp_ctx* c, const int32_t* d_base_perm, int32_t win_start,
                             int32_t win_len, int64_t* d_dist, double* d_obj, cudaStream_t st) {
  const whp_tables T = whp_make_tables(c);
  int32_t rlo, rhi, chi;
  cudaError_t e = launch_window_tables(c, T, d_base_perm, win_start, win_len, &rlo, &rhi, &chi, st);
  if (e != cudaSuccess) return e;
  const int64_t n_nb = (int64_t)win_len * (win_len - 1) / 2;
  int64_t blocks = (n_nb + kSwapWarps - 1) / kSwapWarps;
  const int64_t cap = (int64_t)c->num_sms * 8;
  if (blocks > cap) blocks = cap;
  if (c->swap_stats && (e = cudaMemsetAsync(c->d_swap_stats, 0, 16, st)) != cudaSuccess) return e;
  if (c->swap_stats)
    whp_swaps_kernel<true><<<(unsigned)blocks, kSwapWarps * 32, 0, st>>>(
        T, c->base, win_start, win_len, rlo, rhi, chi, n_nb, d_dist, d_obj, c->d_swap_stats);
  else
    whp_swaps_kernel<false><<<(unsigned)blocks, kSwapWarps * 32, 0, st>>>(
        T, c->base, win_start, win_len, rlo, rhi, chi, n_nb, d_dist, d_obj, nullptr);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t whp_launch_moves(whp_ctx* c, const int32_t* d_base_perm, int32_t win_start,
                             int32_t win_len, int64_t* d_dist, double* d_obj, cudaStream_t st) {
  const whp_tables T = whp_make_tables(c);
  int32_t rlo, rhi, chi;
  cudaError_t e = launch_window_tables(c, T, d_base_perm, win_start, win_len, &rlo, &rhi, &chi, st);
  if (e != cudaSuccess) return e;
  const int64_t n_nb = (int64_t)win_len * (win_len - 1);
  int64_t blocks = (n_nb + kSwapWarps - 1) / kSwapWarps;
  const int64_t cap = (int64_t)c->num_sms * 8;
  if (blocks > cap) blocks = cap;
  if (c->swap_stats && (e = cudaMemsetAsync(c->d_swap_stats, 0, 16, st)) != cudaSuccess) return e;
  if (c->swap_stats)
    whp_moves_kernel<true><<<(unsigned)blocks, kSwapWarps * 32, 0, st>>>(
        T, c->base, win_start, win_len, rlo, rhi, chi, n_nb, d_dist, d_obj, c->d_swap_stats);
  else
    whp_moves_kernel<false><<<(unsigned)blocks, kSwapWarps * 32, 0, st>>>(
        T, c->base, win_start, win_len, rlo, rhi, chi, n_nb, d_dist, d_obj, nullptr);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t whp_launch_apply_move(whp_ctx* c, int32_t* d_base_perm, int32_t win_start,
                                  int32_t win_len, const int64_t* d_idx, cudaStream_t st) {
  whp_apply_move_kernel<<<1, 1, 0, st>>>(d_base_perm, win_start, win_len, d_idx);
  c->launches += 1;
  return cudaGetLastError();
}
