// whp_fast.cu — the tuned candidate path (timed outputs only): three kernels, no cross-lane
// operation inside the inner loops.
//
//   K1 whp_bounds_kernel   one THREAD per candidate runs the next-fit recurrence (D2) over its
//                          permutation row and writes the batch start positions (u16), the
//                          batch count and the batch hash. The order sizes q_o sit in shared
//                          memory as bytes.
//   K2 whp_sets_kernel     one LANE per (candidate, segment): a candidate's batches are cut
//                          into S equal runs; a lane walks the picks of its run one pick per
//                          step. Its occupancy sets are PRIVATE shared-memory words laid out
//                          [word][lane] (bank = lane: never a bank conflict): aisle words hold
//                          16 aisle bits + a batch stamp, class half-words hold an 8-bit visit
//                          count + a batch stamp, so nothing is ever cleared between batches and
//                          r_k (D5) is counted on the fly. Order / pick tables are staged in
//                          shared memory once per block. Per batch: S-shape length (D4) from the
//                          running distinct-aisle count and the max pick record.
//   K3 whp_finish_kernel   one warp per candidate: canonical fp64 penalty (D6), J, outputs.
#include <cstdlib>

#include "whp_walk.cuh"

namespace {

// ---- shared-memory access by 32-bit shared-window address (no generic-address arithmetic) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ uint32_t lds32(uint32_t a) {
  uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v;
}
__device__ __forceinline__ uint32_t lds16(uint32_t a) {
  uint16_t v; asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a)); return v;
}
__device__ __forceinline__ uint32_t lds8(uint32_t a) {
  uint32_t v; asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a)); return v;
}
__device__ __forceinline__ int4 lds128(uint32_t a) {
  int4 v;
  asm volatile("ld.shared.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v));
}
__device__ __forceinline__ void sts16(uint32_t a, uint32_t v) {
  asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"((uint16_t)v));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

// ------------------------------------------------------------------------------------------ K1
constexpr int kBoundsThreads = 64;
constexpr int kRing = 32;  // 16-byte permutation chunks in flight per thread (cp.async ring)

__global__ void __launch_bounds__(kBoundsThreads)
whp_bounds_kernel(const whp_tables T, const int32_t* __restrict__ perms, int64_t n_cand,
                  uint16_t* __restrict__ bpos, int32_t pitch, int32_t* __restrict__ nb_scratch,
                  int32_t* __restrict__ n_batches_out, uint64_t* __restrict__ hash_out,
                  unsigned long long* __restrict__ task_state) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  // [ring: kRing slots x 64 threads x 16 B][sq: q_o as bytes]
  const uint32_t ring0 = smem_u32(smem_raw) + threadIdx.x * 16;
  uint8_t* sq = smem_raw + kRing * kBoundsThreads * 16;
  const uint32_t sq0 = smem_u32(sq);
  for (int i = threadIdx.x; i < T.n_orders; i += kBoundsThreads)
    sq[i] = (uint8_t)(__ldg(T.order_rec + i) & WHP_Q_MASK);
  const int64_t c_raw = (int64_t)blockIdx.x * kBoundsThreads + threadIdx.x;
  const bool have = c_raw < n_cand;
  const int64_t c = have ? c_raw : n_cand - 1;  // idle tail threads redo the last row, no writes
  const int4* __restrict__ row = reinterpret_cast<const int4*>(perms + c * T.n_orders);
  const int n4 = T.n_orders >> 2;
#pragma unroll 1
  for (int k = 0; k < kRing; ++k) {
    if (k < n4) cp_async16(ring0 + k * (kBoundsThreads * 16), row + k);
    cp_async_commit();
  }
  __syncthreads();  // sq visible
  uint16_t* __restrict__ bp = bpos + c * pitch;
  const int C = T.C;
  int load = 0, maxload = 0;
  uint32_t nb = 1;
  uint64_t hash = 1;  // batch 0 starts at position 0: (0+1)*(2*0+1)
  if (have) bp[0] = 0;
  int slot = 0;
#pragma unroll 1
  for (int p4 = 0; p4 < n4; ++p4) {
    cp_async_wait<kRing - 1>();
    const uint32_t slot_addr = ring0 + slot * (kBoundsThreads * 16);
    const int4 v = lds128(slot_addr);
    const int q0 = lds8(sq0 + v.x), q1 = lds8(sq0 + v.y), q2 = lds8(sq0 + v.z), q3 = lds8(sq0 + v.w);
    const int qs[4] = {q0, q1, q2, q3};
    if (p4 + kRing < n4) cp_async16(slot_addr, row + p4 + kRing);
    cp_async_commit();
    slot = (slot + 1) & (kRing - 1);
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      const int load2 = load + qs[t];
      const bool over = load2 > C;
      const uint32_t p = 4u * p4 + t;
      if (over && have) bp[nb] = (uint16_t)p;
      if (over) hash += (uint64_t)(p + 1) * (uint64_t)(2 * nb + 1);
      maxload = over ? max(maxload, load) : maxload;
      nb += over ? 1u : 0u;
      load = over ? qs[t] : load2;
    }
  }
  maxload = __reduce_max_sync(WHP_FULL, max(maxload, load));
  if ((threadIdx.x & 31) == 0) atomicMax(task_state + 1, (unsigned long long)maxload);
  if (!have) return;
  bp[nb] = (uint16_t)T.n_orders;
  nb_scratch[c] = (int32_t)nb;
  if (n_batches_out) n_batches_out[c] = (int32_t)nb;
  if (hash_out) hash_out[c] = hash;
}

// ------------------------------------------------------------------------------------------ K2
struct sets_params {
  int S;         // segments per candidate (power of two <= 32)
  int log2S;
  int cw_words;  // class words per lane  = ceil(K/2)
  int aw_words;  // aisle words per lane  = ceil(NA/16)
  int ring_words;  // per-lane ring of first-pick cursors of the open batch = C + 2
  int warps;     // warps per block
  int64_t n_tasks;  // warp tasks = ceil(n_cand*S/32)
};

// Pick / order tables of K2: staged in shared memory (cursor = 32-bit shared byte address of a
// pick record; the staged order table holds the address of each order's first pick) or read
// from global memory through L1/L2 (cursor = pick index). The pick records K2 reads carry a
// "last pick of its order" flag in bit 8 (d_pick_fast), so no end-of-order cursor is needed.
#define WHP_FAST_LAST 0x100u
constexpr int kIdRing = 4;  // 16-byte order-id chunks in flight per lane (power of two)
template <bool SMEM_TABLES>
struct table_view {
  uint32_t order_base;  // shared address of the staged order table
  const uint32_t* g_order;
  const uint32_t* g_pick;
  __device__ __forceinline__ uint32_t first_pick(uint32_t o) const {
    return SMEM_TABLES ? lds32(order_base + 4 * o) : (__ldg(g_order + o) >> WHP_Q_BITS);
  }
  __device__ __forceinline__ uint32_t pick(uint32_t cur) const {
    return SMEM_TABLES ? lds32(cur) : __ldg(g_pick + cur);
  }
  static constexpr uint32_t kStep = SMEM_TABLES ? 4u : 1u;
};

template <bool SMEM_TABLES, bool DEPOT0>
__global__ void __launch_bounds__(512)
whp_sets_kernel(const whp_tables T, const sets_params P, const uint32_t* __restrict__ pick_fast,
                const int32_t* __restrict__ perms, int64_t n_cand,
                const uint16_t* __restrict__ bpos, int32_t pitch,
                const int32_t* __restrict__ nb_scratch, int64_t* __restrict__ dist_scratch,
                uint32_t* __restrict__ r_scratch, unsigned long long* __restrict__ task_counter) {
  extern __shared__ __align__(16) uint32_t smem[];
  // layout: [order table n_orders][pick table n_items] (if staged) [per-warp private words]
  table_view<SMEM_TABLES> tv;
  tv.g_order = T.order_rec; tv.g_pick = pick_fast; tv.order_base = 0;
  uint32_t* priv = smem;
  uint32_t ring_init = 0;
  if (SMEM_TABLES) {
    const uint32_t pick_base = smem_u32(smem + T.n_orders);
    for (int i = threadIdx.x; i < T.n_orders; i += blockDim.x)
      smem[i] = pick_base + 4 * (__ldg(T.order_rec + i) >> WHP_Q_BITS);
    for (int i = threadIdx.x; i < T.n_items; i += blockDim.x)
      smem[T.n_orders + i] = __ldg(pick_fast + i);
    tv.order_base = smem_u32(smem);
    priv = smem + ((T.n_orders + T.n_items + 31) & ~31);
    ring_init = pick_base;
    __syncthreads();
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int priv_words = (P.cw_words + P.aw_words + P.ring_words + kIdRing * 4) * 32;
  // private words of this lane: word w at my_c[w*32] (bank = lane)
  uint32_t* my_c = priv + (size_t)warp * priv_words + lane;
  const uint32_t cbase = smem_u32(my_c);
  const uint32_t abase = cbase + P.cw_words * 128;
  const uint32_t ring = abase + P.aw_words * 128;
  const uint32_t idring = cbase - lane * 4 + (P.cw_words + P.aw_words + P.ring_words) * 128 + lane * 16;
  for (int w = 0; w < P.ring_words; ++w) sts32(ring + w * 128, ring_init);
  const int Cmax = (int)task_counter[1];  // largest batch load over all candidates (K1) <= T.C
  const int64_t A = T.g.aisle_len;
  const int64_t P2 = 2 * (int64_t)T.g.aisle_spacing;
  const int n4 = T.n_orders >> 2;

  __shared__ unsigned long long s_task[16];
  for (;;) {
    // claim the next warp task (32 consecutive (candidate, segment) pairs)
    if (lane == 0) s_task[warp] = atomicAdd(task_counter, 1ull);
    __syncwarp();
    const int64_t task = (int64_t)s_task[warp];
    __syncwarp();
    if (task >= P.n_tasks) break;
    const int64_t unit = task * 32 + lane;
    const int64_t cand_raw = unit >> P.log2S;
    const int seg = (int)(unit & (P.S - 1));
    const bool have = cand_raw < n_cand;
    const int64_t cand = have ? cand_raw : n_cand - 1;
    int b_lo = 0, b_hi = 0;
    if (have) {
      const int nb = __ldg(nb_scratch + cand);
      b_lo = (int)((int64_t)seg * nb >> P.log2S);
      b_hi = (int)((int64_t)(seg + 1) * nb >> P.log2S);
    }
    const int nbseg = b_hi - b_lo;
    const int nbmax = __reduce_max_sync(WHP_FULL, nbseg);
    // clear the private set words (stamp 0 is older than every live batch)
    for (int w = 0; w < P.cw_words + P.aw_words; ++w) my_c[w * 32] = 0;
    const uint16_t* __restrict__ bp = bpos + cand * pitch + b_lo;
    const int4* __restrict__ row4 = reinterpret_cast<const int4*>(perms + cand * T.n_orders);
    // ---- order-id stream of this lane: positions from the segment start on. The row is
    // streamed through a private cp.async ring of kIdRing 16-byte chunks ([slot][lane] x 16 B),
    // so global latency never sits on the critical path.
    int p_next = (int)__ldg(bp);
    int pe_ahead = (nbseg > 0) ? (int)__ldg(bp + 1) : p_next;  // boundary loaded one batch early
    int vi = p_next >> 2;  // next chunk to consume
#pragma unroll
    for (int k = 0; k < kIdRing; ++k) {
      cp_async16(idring + ((vi + k) & (kIdRing - 1)) * 512, row4 + min(vi + k, n4 - 1));
      cp_async_commit();
    }
    cp_async_wait<kIdRing - 1>();
    int4 va = lds128(idring + (vi & (kIdRing - 1)) * 512);
    cp_async16(idring + (vi & (kIdRing - 1)) * 512, row4 + min(vi + kIdRing, n4 - 1));
    cp_async_commit();
    ++vi;
    int vleft = 4 - (p_next & 3);
    for (int k = p_next & 3; k > 0; --k) { va.x = va.y; va.y = va.z; va.z = va.w; }

    int64_t D = 0;
    for (int j = 0; j < nbmax; ++j) {
      int left = 0;  // orders of batch j
      if (j < nbseg) {
        left = pe_ahead - p_next;
        p_next = pe_ahead;
        if (j + 1 < nbseg) pe_ahead = (int)__ldg(bp + j + 2);
      }
      const bool live = left > 0;
      // ---- prefill the private ring with the first-pick cursor of every order of the batch
      const int maxleft = __reduce_max_sync(WHP_FULL, left);
      for (int k = 0; k < maxleft; ++k) {
        if (k < left) {
          const uint32_t o = (uint32_t)va.x;
          va.x = va.y; va.y = va.z; va.z = va.w;
          if (--vleft == 0) {
            const uint32_t slot = idring + (vi & (kIdRing - 1)) * 512;
            cp_async_wait<kIdRing - 1>();
            va = lds128(slot);
            cp_async16(slot, row4 + min(vi + kIdRing, n4 - 1));
            cp_async_commit();
            ++vi;
            vleft = 4;
          }
          sts32(ring + k * 128, tv.first_pick(o));
        }
      }
      const uint32_t stamp = (uint32_t)(j + 1);
      const uint32_t stamp_hi = stamp << 16, stamp_c = stamp << 8, stamp_c1 = stamp_c + 1;
      uint32_t kmax = 0, kmin = 0xffffffffu;
      int m = 0;
      uint32_t cur = lds32(ring);
      uint32_t n_cur = lds32(ring + 128);
      uint32_t rp = ring + 256;
      uint32_t rec = tv.pick(cur);
#pragma unroll 1
      for (int t = 0; t < Cmax; ++t) {
        if (left > 0) {
          // cursor of the next step's pick: next record, or the next order's first pick
          uint32_t nxt = cur + table_view<SMEM_TABLES>::kStep;
          if (rec & WHP_FAST_LAST) {
            nxt = n_cur;
            n_cur = lds32(rp);
            rp += 128;
            --left;
          }
          cur = nxt;
          const uint32_t rec_next = tv.pick(cur);
          // ---- this step's pick
          kmax = max(kmax, rec);
          if (!DEPOT0) kmin = min(kmin, rec);
          const uint32_t aaddr = abase + ((rec >> 26) << 7);
          uint32_t bit;  // 1 << (a_lo): funnel shift uses (rec >> 21) mod 32 = a_lo (spacer bit)
          asm("shf.l.wrap.b32 %0, %1, %2, %3;" : "=r"(bit) : "r"(0u), "r"(1u), "r"(rec >> 21));
          const uint32_t x = max(lds32(aaddr), stamp_hi);  // an older stamp compares lower: empty
          const uint32_t x2 = x | bit;
          if (x2 != x) ++m;
          sts32(aaddr, x2);
          const uint32_t caddr = cbase + (((rec << 6) & 0x3f80u) | ((rec << 1) & 2u));
          const uint32_t y = lds16(caddr);  // stamp:8 | visit count:8
          if (y < stamp_c) sts16(caddr, (y & 0xffu) + stamp_c1);
          rec = rec_next;
        }
      }
      if (live) {  // D4
        const int64_t a_max = WHP_PICK_AISLE(kmax);
        const int64_t d_last =
            (int64_t)((kmax >> WHP_PICK_SLOT_SHIFT) & WHP_PICK_SLOT_MASK) * T.g.slot_pitch;
        int64_t H;
        if (DEPOT0) {
          H = P2 * a_max;
        } else {
          const int64_t a_min = WHP_PICK_AISLE(kmin), a0 = T.g.depot_aisle;
          H = (int64_t)T.g.aisle_spacing * (llabs(a0 - a_min) + (a_max - a_min) + llabs(a_max - a0));
        }
        D += H + ((m & 1) ? (int64_t)(m - 1) * A + 2 * d_last : (int64_t)m * A);
      }
    }
    // combine the S segment lanes of each candidate: D and the class visit counts
#pragma unroll
    for (int o = 1; o < 32; o <<= 1)
      if (o < P.S) D += __shfl_xor_sync(WHP_FULL, D, o);
    if (have && seg == 0) dist_scratch[cand] = D;
    uint32_t* __restrict__ rrow = r_scratch + cand * P.cw_words;
    for (int w = 0; w < P.cw_words; ++w) {
      uint32_t cnt = my_c[w * 32] & 0x00ff00ffu;  // two 16-bit counts
      for (int o = 1; o < P.S; o <<= 1) cnt += __shfl_xor_sync(WHP_FULL, cnt, o);
      if (have && seg == 0) rrow[w] = cnt;
    }
    __syncwarp();
  }
}

// ------------------------------------------------------------------------------------------ K3
__global__ void __launch_bounds__(256)
whp_finish_kernel(const whp_tables T, int64_t n_cand, const int64_t* __restrict__ dist_scratch,
                  const uint16_t* __restrict__ r_scratch, int32_t r_pitch,
                  int64_t* __restrict__ dist, double* __restrict__ penalty,
                  double* __restrict__ obj) {
  const int lane = threadIdx.x & 31;
  const int64_t cand = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (cand >= n_cand) return;
  const uint16_t* __restrict__ r = r_scratch + cand * r_pitch;
  double s = 0.0;
  for (int k = lane; k < T.K; k += 32) {  // same canonical order as whp_penalty (D6)
    const double c = __dsub_rn(__ldg(T.tvw + k), (double)__ldg(r + k));
    const double u = __dmul_rn(__ldg(T.tvw + 2 * T.K + k), c);
    const double term = __dadd_rn(__dmul_rn(__ldg(T.tvw + T.K + k), c), __dmul_rn(u, u));
    s = __dadd_rn(s, term);
  }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) s = __dadd_rn(s, __shfl_xor_sync(WHP_FULL, s, off));
  if (lane == 0) {
    const int64_t D = dist_scratch[cand];
    if (dist) dist[cand] = D;
    if (penalty) penalty[cand] = s;
    if (obj) obj[cand] = __dadd_rn((double)D, s);
  }
}

}  // namespace

// nb <= 2*n_items/(C+1) + 1: consecutive next-fit batches together hold more than C items
static int64_t nb_upper_bound(const whp_ctx* c) {
  int64_t ub = 2ll * c->n_items / ((int64_t)c->C + 1) + 1;
  return ub < c->n_orders ? ub : c->n_orders;
}

bool whp_fast_eligible(const whp_ctx* c) {
  if (c->n_orders % 4 != 0 || c->n_orders >= 65536) return false;
  if ((nb_upper_bound(c) + 31) / 32 > 255) return false;  // 8-bit stamps, S <= 32
  if (c->n_orders > 160 * 1024) return false;              // q bytes in shared memory (K1)
  if (c->C > 64) return false;                             // per-lane cursor ring of C+2 words
  return true;
}

cudaError_t whp_launch_eval_fast(whp_ctx* c, const int32_t* d_perms, int64_t n_cand,
                                 const whp_eval_out& out, cudaStream_t st) {
  const whp_tables T = whp_make_tables(c);
  const int64_t nb_ub = nb_upper_bound(c);
  const int32_t pitch = (int32_t)((nb_ub + 1 + 7) & ~7ll);
  const int cw_words = (c->K + 1) / 2, aw_words = (c->g.n_aisles + 15) / 16;
  // scratch (grow-only)
  if (c->fast_cap < n_cand || c->fast_pitch != pitch) {
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    cudaFree(c->d_bpos); cudaFree(c->d_nb); cudaFree(c->d_dist_scratch); cudaFree(c->d_r_scratch);
    c->d_bpos = nullptr; c->d_nb = nullptr; c->d_dist_scratch = nullptr; c->d_r_scratch = nullptr;
    c->fast_cap = 0;
    if ((e = cudaMalloc(&c->d_bpos, sizeof(uint16_t) * (size_t)n_cand * pitch)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_nb, sizeof(int32_t) * (size_t)n_cand)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_dist_scratch, sizeof(int64_t) * (size_t)n_cand)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_r_scratch, sizeof(uint32_t) * (size_t)n_cand * cw_words)) != cudaSuccess) return e;
    c->fast_cap = n_cand; c->fast_pitch = pitch;
  }
  // K1
  {
    cudaError_t e0 = cudaMemsetAsync(c->d_task, 0, 2 * sizeof(unsigned long long), st);
    if (e0 != cudaSuccess) return e0;
    const size_t smem = (size_t)kRing * kBoundsThreads * 16 + (size_t)c->n_orders;
    static bool attr_done = false;
    if (!attr_done) {
      cudaFuncSetAttribute(whp_bounds_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
      attr_done = true;
    }
    const unsigned blocks = (unsigned)((n_cand + kBoundsThreads - 1) / kBoundsThreads);
    whp_bounds_kernel<<<blocks, kBoundsThreads, smem, st>>>(T, d_perms, n_cand, c->d_bpos, pitch,
                                                            c->d_nb, out.n_batches, out.batch_hash,
                                                            c->d_task);
    c->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  // K2
  {
    cudaError_t e;
    const size_t table_bytes = 4 * (((size_t)c->n_orders + c->n_items + 31) & ~(size_t)31);
    const int ring_words = c->C + 2;
    const size_t priv_per_warp = (size_t)(cw_words + aw_words + ring_words + kIdRing * 4) * 128;
    const size_t smem_max = (size_t)c->smem_optin - 1024;
    bool smem_tables = table_bytes + 4 * priv_per_warp <= smem_max;
    const size_t avail = smem_max - (smem_tables ? table_bytes : 0);
    int warps = (int)(avail / priv_per_warp);
    if (warps > 16) warps = 16;
    if (warps < 1) return cudaErrorInvalidConfiguration;
    int blocks_per_sm = 1;
    if (!smem_tables) {  // small private footprint: several blocks per SM
      const size_t per_block = priv_per_warp * warps;
      blocks_per_sm = (int)(smem_max / (per_block + 1024));
      if (blocks_per_sm > 4) blocks_per_sm = 4;
      if (blocks_per_sm < 1) blocks_per_sm = 1;
    }
    const int64_t resident_warps = (int64_t)c->num_sms * blocks_per_sm * warps;
    // segments: enough for the 8-bit stamps, and ~4 warp tasks per resident warp
    int S = 1;
    while (S < 32 && ((nb_ub + S - 1) / S > 255 || n_cand * S < 4 * resident_warps * 32)) S <<= 1;
    if (const char* e = getenv("WHP_SEGMENTS")) { int v = atoi(e); if (v >= 1 && v <= 32 && (v & (v - 1)) == 0 && (nb_ub + v - 1) / v <= 255) S = v; }
    sets_params P;
    P.S = S; P.log2S = 0; while ((1 << P.log2S) < S) ++P.log2S;
    P.cw_words = cw_words; P.aw_words = aw_words; P.ring_words = ring_words; P.warps = warps;
    P.n_tasks = (n_cand * S + 31) / 32;
    int64_t blocks = (P.n_tasks + warps - 1) / warps;
    if (blocks > (int64_t)c->num_sms * blocks_per_sm) blocks = (int64_t)c->num_sms * blocks_per_sm;
    const size_t smem = (smem_tables ? table_bytes : 0) + priv_per_warp * warps;
    const bool depot0 = c->g.depot_aisle == 0;
#define WHP_LAUNCH_SETS(ST, D0)                                                                  \
  do {                                                                                           \
    cudaFuncSetAttribute(whp_sets_kernel<ST, D0>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                         (int)smem_max);                                                         \
    whp_sets_kernel<ST, D0><<<(unsigned)blocks, warps * 32, smem, st>>>(                          \
        T, P, c->d_pick_fast, d_perms, n_cand, c->d_bpos, pitch, c->d_nb, c->d_dist_scratch, c->d_r_scratch,     \
        c->d_task);                                                                              \
  } while (0)
    if (smem_tables && depot0) WHP_LAUNCH_SETS(true, true);
    else if (smem_tables) WHP_LAUNCH_SETS(true, false);
    else if (depot0) WHP_LAUNCH_SETS(false, true);
    else WHP_LAUNCH_SETS(false, false);
#undef WHP_LAUNCH_SETS
    c->launches += 1;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  // K3
  if (out.dist || out.penalty || out.obj) {
    const unsigned blocks = (unsigned)((n_cand * 32 + 255) / 256);
    whp_finish_kernel<<<blocks, 256, 0, st>>>(T, n_cand, c->d_dist_scratch,
                                              (const uint16_t*)c->d_r_scratch, 2 * cw_words,
                                              out.dist, out.penalty, out.obj);
    c->launches += 1;
    return cudaGetLastError();
  }
  return cudaSuccess;
}
