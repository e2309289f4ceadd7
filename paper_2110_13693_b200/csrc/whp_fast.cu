// whp_fast.cu — the tuned candidate path (timed outputs and r_k): three kernels with no
// cross-lane operation inside the inner loops.
//
//   K1 whp_bounds_kernel   one THREAD per candidate runs the next-fit recurrence (D2) over its
//                          permutation row (streamed through a cp.async ring) and writes (i) a
//                          bitmask of batch-start positions, (ii) the batch count, (iii) the
//                          "cursor stream": for every position the 16-bit index of the order's
//                          first pick record, so K2 needs neither the permutation nor the order
//                          table.
//   K2 whp_sets_kernel     one LANE per (candidate, segment): a candidate's batches are cut into
//                          S equal runs; a lane walks the picks of its run, one pick per step.
//                          Its occupancy sets are PRIVATE shared-memory words laid out
//                          [word][lane] (bank = lane: never a bank conflict); a word holds 16
//                          set bits plus a 16-bit batch stamp, so an unsigned max() with
//                          (stamp << 16) empties a stale word and nothing is ever cleared.
//                          Per batch: S-shape length (D4) from the running distinct-aisle count
//                          and the max pick record; the batch's class set is added into
//                          bit-sliced ("vertical") counters held in registers (D5).
//   K3 whp_finish_kernel   one warp per candidate: decodes the vertical counters into r_k,
//                          canonical fp64 penalty (D6), J, outputs.
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
__device__ __forceinline__ int4 lds128(uint32_t a) {
  int4 v;
  asm volatile("ld.shared.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v));
}
// if (k < n) st.shared [a] = v — predicated, never a branch
__device__ __forceinline__ void sts32_if_lt(uint32_t k, uint32_t n, uint32_t a, uint32_t v) {
  asm volatile("{ .reg .pred pq; setp.lt.u32 pq, %0, %1; @pq st.shared.u32 [%2], %3; }" ::"r"(k), "r"(n), "r"(a), "r"(v));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }
// 1 << (n mod 32): the funnel shift wraps its shift amount, so no mask instruction is needed
__device__ __forceinline__ uint32_t one_shl_wrap(uint32_t n) {
  uint32_t r; asm("shf.l.wrap.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(0u), "r"(1u), "r"(n)); return r;
}

// ------------------------------------------------------------------------------------------ K1
constexpr int kBoundsThreads = 64;
constexpr int kRing = 32;  // 16-byte permutation chunks in flight per thread (cp.async ring)

__global__ void __launch_bounds__(kBoundsThreads)
whp_bounds_kernel(const uint32_t* __restrict__ order_fast, int32_t n_orders, int32_t C,
                  const int32_t* __restrict__ perms, int64_t n_cand,
                  uint32_t* __restrict__ bmask, int32_t bm_pitch, uint16_t* __restrict__ cstream,
                  int32_t cs_pitch, int32_t* __restrict__ nb_scratch,
                  int32_t* __restrict__ n_batches_out) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  // [ring: kRing slots x 64 threads x 16 B][order_fast: (cursor << 8 | q) per order]
  const uint32_t ring0 = smem_u32(smem_raw) + threadIdx.x * 16;
  uint32_t* sorec = reinterpret_cast<uint32_t*>(smem_raw + kRing * kBoundsThreads * 16);
  const uint32_t sorec0 = smem_u32(sorec);
  for (int i = threadIdx.x; i < n_orders; i += kBoundsThreads) sorec[i] = __ldg(order_fast + i);
  const int64_t c = (int64_t)blockIdx.x * kBoundsThreads + threadIdx.x;
  const bool have = c < n_cand;
  const int4* __restrict__ row = reinterpret_cast<const int4*>(perms + (have ? c : 0) * n_orders);
  const int n4 = n_orders >> 2;
  if (have) {
#pragma unroll 1
    for (int k = 0; k < kRing; ++k) {
      if (k < n4) cp_async16(ring0 + k * (kBoundsThreads * 16), row + k);
      else asm volatile("st.shared.v4.u32 [%0], {%1,%1,%1,%1};" ::"r"(ring0 + k * (kBoundsThreads * 16)), "r"(0u));
      cp_async_commit();
    }
  }
  __syncthreads();  // sorec visible
  if (!have) return;
  uint32_t* __restrict__ bm = bmask + c * bm_pitch;
  uint2* __restrict__ cs = reinterpret_cast<uint2*>(cstream + c * cs_pitch);
  const int nw = (n_orders + 31) >> 5;
  // Next-fit recurrence on room = C - load, one dependent instruction per position:
  //   room' = umin(room - q, C - q)   (room < q wraps room - q above C - q: a new batch opens)
  uint32_t room = (uint32_t)C;
  uint32_t nb = 0;
  int p4 = 0, slot = 0;
  // 3-stage software pipeline, one chunk (4 positions) per stage: (A) order ids of chunk i+2
  // leave the cp.async ring, (B) their order records are gathered for chunk i+1, (C) chunk i
  // runs the next-fit recurrence — the only loop-carried dependency chain.
  int4 ids = make_int4(0, 0, 0, 0);
  uint32_t rb[4] = {0, 0, 0, 0}, rc[4] = {0, 0, 0, 0};
  auto stage_a = [&](int chunk) {  // chunk may run past the row end: the slot is then stale
    cp_async_wait<kRing - 1>();
    const uint32_t slot_addr = ring0 + slot * (kBoundsThreads * 16);
    const int4 v = lds128(slot_addr);
    if (chunk + kRing < n4) cp_async16(slot_addr, row + chunk + kRing);
    cp_async_commit();
    slot = (slot + 1) & (kRing - 1);
    return v;
  };
  auto stage_b = [&](const int4& v, uint32_t (&r)[4]) {
    // ids past the row end are stale ring contents (ids of earlier chunks, or the zero fill):
    // always valid order ids, so the gather stays in the table
    r[0] = lds32(sorec0 + 4 * v.x); r[1] = lds32(sorec0 + 4 * v.y);
    r[2] = lds32(sorec0 + 4 * v.z); r[3] = lds32(sorec0 + 4 * v.w);
  };
  ids = stage_a(0);
  stage_b(ids, rc);
  ids = stage_a(1);
  stage_b(ids, rb);
  ids = stage_a(2);
#pragma unroll 1
  for (int w = 0; w < nw; ++w) {
    uint32_t bits = (w == 0) ? 1u : 0u;  // batch 0 starts at position 0
#pragma unroll
    for (int k = 0; k < 8; ++k, ++p4) {
      if (p4 < n4) {
        uint32_t rn[4];
        stage_b(ids, rn);        // chunk p4 + 2
        ids = stage_a(p4 + 3);
        // cursor stream: 4 x u16 = bits 8..23 of the order records
        cs[p4] = make_uint2(__byte_perm(rc[0], rc[1], 0x6521), __byte_perm(rc[2], rc[3], 0x6521));
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const uint32_t q = rc[t] & WHP_Q_MASK;
          const bool over = room < q;
          room = min(room - q, (uint32_t)C - q);
          if (over) bits |= 1u << (4 * k + t);
          rc[t] = rb[t];
          rb[t] = rn[t];
        }
      }
    }
    nb += __popc(bits);
    if (w == (n_orders >> 5)) bits |= 1u << (n_orders & 31);  // end sentinel in a partial word
    bm[w] = bits;
  }
  if ((n_orders & 31) == 0) bm[nw] = 1u;  // end sentinel in a word of its own
  nb_scratch[c] = (int32_t)nb;
  if (n_batches_out) n_batches_out[c] = (int32_t)nb;
}

// ------------------------------------------------------------------------------------------ K2
constexpr int kMaxPlanes = 8;  // vertical counter bit planes: up to 255 batches per segment
#define WHP_FAST_LAST 0x100u

struct sets_params {
  int S;           // segments per candidate (power of two <= 32)
  int log2S;
  int aw_words;    // aisle words per lane  = ceil(NA/16)
  int ring_words;  // per-lane ring of first-pick cursors of the open batch = C + 2
  int id_slots;    // 16-byte cursor-stream chunks resident per lane (power of two, covers a batch)
  int bm_pitch, cs_pitch;
  int n_items_pad;
  int64_t n_tasks;  // warp tasks = ceil(n_cand*S/32)
};

template <bool SMEM_TABLES, bool DEPOT0, int KW, int kPlanes>
__global__ void __launch_bounds__(512, 1)
whp_sets_kernel(const whp_tables T, const sets_params P, const uint32_t* __restrict__ pick_fast,
                const uint16_t* __restrict__ cstream, const uint32_t* __restrict__ bmask,
                const int32_t* __restrict__ nb_scratch, int64_t n_cand,
                int64_t* __restrict__ dist_scratch, uint32_t* __restrict__ planes_out,
                uint64_t* __restrict__ hash_out, unsigned long long* __restrict__ task_counter) {
  extern __shared__ __align__(16) uint32_t smem[];
  // layout: [pick table n_items_pad] (if staged) [per-warp private words]
  constexpr int CW = 2 * KW;  // 16-bit stamped class words per lane
  uint32_t* priv = smem;
  uint32_t pick_base = 0;
  if (SMEM_TABLES) {
    for (int i = threadIdx.x; i < P.n_items_pad; i += blockDim.x) smem[i] = __ldg(pick_fast + i);
    pick_base = smem_u32(smem);
    priv = smem + ((P.n_items_pad + 31) & ~31);
    __syncthreads();
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int priv_words = (CW + P.aw_words + P.ring_words + P.id_slots * 4) * 32;
  // private words of this lane: word w at my_c[w*32] (bank = lane)
  uint32_t* my_c = priv + (size_t)warp * priv_words + lane;
  const uint32_t cbase = smem_u32(my_c);
  const uint32_t abase = cbase + CW * 128;
  const uint32_t ring = abase + P.aw_words * 128;
  const uint32_t idring = cbase - lane * 4 + (CW + P.aw_words + P.ring_words) * 128 + lane * 16;
  for (int w = 0; w < P.ring_words; ++w) sts32(ring + w * 128, pick_base);
  const int Cmax = T.C;
  const int64_t A = T.g.aisle_len;
  const int64_t P2 = 2 * (int64_t)T.g.aisle_spacing;
  const int n8 = P.cs_pitch >> 3;  // 16-byte chunks per cursor-stream row

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
    for (int w = 0; w < CW + P.aw_words; ++w) my_c[w * 32] = 0;
    uint32_t pl[kPlanes][KW];
#pragma unroll
    for (int p = 0; p < kPlanes; ++p)
#pragma unroll
      for (int w = 0; w < KW; ++w) pl[p][w] = 0;

    // ---- locate the first batch of the segment in the boundary bitmask (select b_lo)
    const uint32_t* __restrict__ bm = bmask + cand * P.bm_pitch;
    int wi = 0;
    uint32_t bw = __ldg(bm);
    if (nbseg > 0) {
      int acc = 0;
      for (;;) {
        const int pc = __popc(bw);
        if (acc + pc > b_lo) break;
        acc += pc;
        ++wi;
        bw = __ldg(bm + wi);
      }
      for (int r = b_lo - acc; r > 0; --r) bw &= bw - 1;  // drop the starts before mine
    }
    uint32_t bw_next = __ldg(bm + min(wi + 1, P.bm_pitch - 1));
    int p = 32 * wi + __ffs(bw) - 1;  // first position of the segment

    // ---- cursor stream of this lane through a private cp.async ring ([slot][lane] x 16 B):
    // chunk c (cursors of positions 8c..8c+7) lives in slot c mod kIdRing
    const uint4* __restrict__ cs = reinterpret_cast<const uint4*>(cstream + cand * P.cs_pitch);
    {
      const int c0 = p >> 3;
      for (int k = 0; k < P.id_slots; ++k)
        cp_async16(idring + ((c0 + k) & (P.id_slots - 1)) * 512, cs + min(c0 + k, n8 - 1));
      cp_async_commit();
    }

    int64_t D = 0;
    uint64_t hash = 0;
    for (int j = 0; j < nbmax; ++j) {
      int left = 0;  // orders of batch j
      if (j < nbseg) {
        bw &= bw - 1;  // past my own start bit: the next set bit is the next batch (or the end)
        while (bw == 0) {
          ++wi;
          bw = bw_next;
          bw_next = __ldg(bm + min(wi + 1, P.bm_pitch - 1));
        }
        const int pe = 32 * wi + __ffs(bw) - 1;
        hash += (uint64_t)(uint32_t)(p + 1) * (uint64_t)(uint32_t)(2 * (b_lo + j) + 1);
        left = pe - p;
        p = pe;
      }
      const bool live = left > 0;
      // ---- prefill the private ring with the first-pick cursor of every order of the batch,
      // one 16-byte chunk (8 positions) of the cursor stream at a time
      const int p0 = p - left;                       // first position of the batch
      const int nc = live ? ((p - 1) >> 3) - (p0 >> 3) + 1 : 0;   // chunks the batch touches
      const int nf = (p >> 3) - (p0 >> 3);           // chunks the batch finishes
      const int ncmax = __reduce_max_sync(WHP_FULL, nc);
      cp_async_wait<0>();  // issued a whole batch ago: normally complete already
      for (int i = 0; i < ncmax; ++i) {
        if (i < nc) {
          const int c = (p0 >> 3) + i;
          const int4 v = lds128(idring + (c & (P.id_slots - 1)) * 512);
          const int kb = 8 * c - p0;               // ring index of the chunk's first cursor
          const uint32_t rb = ring + kb * 128;
          const uint32_t vv[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            const uint32_t c16 = (e & 1) ? (vv[e >> 1] >> 16) : (vv[e >> 1] & 0xffffu);
            sts32_if_lt((uint32_t)(kb + e), (uint32_t)left, rb + e * 128,
                        SMEM_TABLES ? pick_base + 8 * c16 : 2 * c16);
          }
        }
      }
      {  // refill the slots of the finished chunks; they land while the batch is processed
        const int nfmax = __reduce_max_sync(WHP_FULL, nf);
        for (int i = 0; i < nfmax; ++i)
          if (i < nf) {
            const int c = (p0 >> 3) + i;
            cp_async16(idring + (c & (P.id_slots - 1)) * 512, cs + min(c + P.id_slots, n8 - 1));
          }
        cp_async_commit();
      }
      const uint32_t stamp_hi = (uint32_t)(j + 1) << 16;
      uint32_t kmax = 0, kmin = 0xffffffffu;
      int m = 0;
      uint32_t cur = lds32(ring);
      uint32_t n_cur = lds32(ring + 128);
      uint32_t rp = ring + 256;
      const uint32_t rp_end = rp + 128 * max(left - 1, 0);  // left-1 moves to a next order
      uint32_t rec = SMEM_TABLES ? lds32(cur) : __ldg(pick_fast + cur);
      // Branch-free step: every lane runs Cmax steps. A lane that has finished its batch stays
      // on the batch's final pick and re-inserts it (set inserts and max are idempotent); a
      // lane without a batch walks to the end of order 0 and stays there — its sets are
      // discarded at the close below.
#pragma unroll 2
      for (int t = 0; t < Cmax; ++t) {
        // cursor of the next step's pick: next record, the next order's first pick, or stay
        uint32_t nxt = cur + (SMEM_TABLES ? 4u : 1u);
        const bool last = (rec & WHP_FAST_LAST) != 0;
        const bool more = last && (rp != rp_end);
        if (last) nxt = cur;
        if (more) {
          nxt = n_cur;
          n_cur = lds32(rp);
          rp += 128;
        }
        cur = nxt;
        const uint32_t rec_next = SMEM_TABLES ? lds32(cur) : __ldg(pick_fast + cur);
        // ---- this step's pick
        kmax = max(kmax, rec);
        if (!DEPOT0) kmin = min(kmin, rec);
        const uint32_t aaddr = abase + ((rec >> 26) << 7);
        const uint32_t abit = one_shl_wrap(rec >> 21);  // spacer bit: (rec >> 21) mod 32 = a_lo
        const uint32_t x = max(lds32(aaddr), stamp_hi);  // an older stamp compares lower: empty
        const uint32_t x2 = x | abit;
        asm("{ .reg .pred pp; setp.ne.u32 pp, %1, %2; @pp add.s32 %0, %0, 1; }" : "+r"(m) : "r"(x2), "r"(x));
        sts32(aaddr, x2);
        const uint32_t caddr = cbase + ((rec & 0xf0u) << 3);
        const uint32_t cbit = one_shl_wrap(rec & 15u);
        const uint32_t y = max(lds32(caddr), stamp_hi);
        sts32(caddr, y | cbit);
        rec = rec_next;
      }
      // ---- close the batch: D4, and the class set into the vertical counters (D5)
      if (live) {
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
#pragma unroll
      for (int w = 0; w < KW; ++w) {
        // lanes without a batch j ran the steps on a dummy pick: their set is discarded
        const uint32_t y0 = max(lds32(cbase + (2 * w) * 128), stamp_hi);
        const uint32_t y1 = max(lds32(cbase + (2 * w + 1) * 128), stamp_hi);
        uint32_t carry = live ? __byte_perm(y0, y1, 0x5410) : 0u;  // 32 class bits of this batch
#pragma unroll
        for (int pp = 0; pp < kPlanes; ++pp) {
          const uint32_t t2 = pl[pp][w] & carry;
          pl[pp][w] ^= carry;
          carry = t2;
        }
      }
    }
    // ---- combine the S segment lanes of each candidate (D, hash); write the counters
#pragma unroll
    for (int o = 1; o < 32; o <<= 1)
      if (o < P.S) {
        D += __shfl_xor_sync(WHP_FULL, D, o);
        hash += __shfl_xor_sync(WHP_FULL, hash, o);
      }
    if (have && seg == 0) {
      dist_scratch[cand] = D;
      if (hash_out) hash_out[cand] = hash;
    }
    // bit-sliced addition of the S lanes' vertical counters (one more plane per level)
    {
      uint32_t* __restrict__ po = planes_out + cand * ((kMaxPlanes + 5) * KW);
#pragma unroll
      for (int w = 0; w < KW; ++w) {
        uint32_t a[kPlanes + 5];
#pragma unroll
        for (int pp = 0; pp < kPlanes + 5; ++pp) a[pp] = pp < kPlanes ? pl[pp][w] : 0u;
#pragma unroll
        for (int lvl = 0; lvl < 5; ++lvl) {
          if ((1 << lvl) < P.S) {
            uint32_t carry = 0;
#pragma unroll
            for (int pp = 0; pp < kPlanes + lvl; ++pp) {
              const uint32_t b = __shfl_xor_sync(WHP_FULL, a[pp], 1 << lvl);
              const uint32_t sum = a[pp] ^ b ^ carry;
              carry = (a[pp] & b) | (carry & (a[pp] ^ b));
              a[pp] = sum;
            }
            a[kPlanes + lvl] = carry;
          }
        }
        if (have && seg == 0) {
#pragma unroll
          for (int pp = 0; pp < kPlanes + 5; ++pp)
            if (pp < kPlanes + P.log2S) po[pp * KW + w] = a[pp];
        }
      }
    }
    __syncwarp();
  }
}

// ------------------------------------------------------------------------------------------ K3
// one warp per candidate; lane l owns classes l, l+32, ... in ascending order — exactly the
// canonical 32-lane accumulation of D6.
__global__ void __launch_bounds__(256)
whp_finish_kernel(const whp_tables T, int64_t n_cand, const int64_t* __restrict__ dist_scratch,
                  const uint32_t* __restrict__ planes, int KW, int planes_used,
                  int64_t* __restrict__ dist, double* __restrict__ penalty,
                  double* __restrict__ obj, int32_t* __restrict__ resp) {
  const int lane = threadIdx.x & 31;
  const int64_t cand = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (cand >= n_cand) return;
  // the candidate's (kMaxPlanes+5) x KW counter words, one coalesced read, then warp broadcasts
  const uint32_t* __restrict__ pc = planes + cand * ((kMaxPlanes + 5) * KW);
  const int total = planes_used * KW;  // <= 13 * 8 = 104
  uint32_t regs[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) regs[i] = (lane + 32 * i < total) ? __ldg(pc + lane + 32 * i) : 0u;
  double s = 0.0;
  const int kw_used = (T.K + 31) >> 5;
  for (int w = 0; w < kw_used; ++w) {
    int r = 0;
    for (int pp = 0; pp < planes_used; ++pp) {
      const int idx = pp * KW + w;
      const int hi = idx >> 5;
      const uint32_t src = hi == 0 ? regs[0] : hi == 1 ? regs[1] : hi == 2 ? regs[2] : regs[3];
      const uint32_t word = __shfl_sync(WHP_FULL, src, idx & 31);
      r += (int)((word >> lane) & 1u) << pp;
    }
    const int k = 32 * w + lane;
    if (k < T.K) {
      if (resp) resp[cand * T.K + k] = r;
      const double c = __dsub_rn(__ldg(T.tvw + k), (double)r);
      const double u = __dmul_rn(__ldg(T.tvw + 2 * T.K + k), c);
      const double term = __dadd_rn(__dmul_rn(__ldg(T.tvw + T.K + k), c), __dmul_rn(u, u));
      s = __dadd_rn(s, term);
    }
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
  if (!c->fast_tables_ok) return false;                       // cursors must fit 16 bits
  if (c->n_orders % 4 != 0 || c->n_orders >= 65536) return false;
  if ((nb_upper_bound(c) + 31) / 32 > 255) return false;      // 8 counter planes, S <= 32
  if (c->C > 64) return false;                                // per-lane cursor ring of C+2 words
  if ((size_t)kRing * kBoundsThreads * 16 + 4 * (size_t)c->n_orders > (size_t)c->smem_optin - 1024)
    return false;                                             // K1: order table in shared memory
  return true;
}

cudaError_t whp_launch_eval_fast(whp_ctx* c, const int32_t* d_perms, int64_t n_cand,
                                 const whp_eval_out& out, cudaStream_t st) {
  const whp_tables T = whp_make_tables(c);
  const int64_t nb_ub = nb_upper_bound(c);
  const int32_t bm_pitch = (int32_t)((((c->n_orders + 31) >> 5) + 2 + 3) & ~3);
  const int32_t cs_pitch = (int32_t)((c->n_orders + 7) & ~7);
  const int KW = c->K <= 32 ? 1 : c->K <= 64 ? 2 : c->K <= 128 ? 4 : c->K <= 224 ? 7 : 8;
  const int aw_words = (c->g.n_aisles + 15) / 16;
  const int ring_words = c->C + 2;
  int id_slots = 4;  // a batch of C orders touches at most (C+14)/8 chunks
  while (id_slots < (c->C + 14) / 8 + 1) id_slots <<= 1;
  // K2 shape
  const size_t table_bytes = 4 * (((size_t)c->n_items_pad + 31) & ~(size_t)31);
  const size_t priv_per_warp = (size_t)(2 * KW + aw_words + ring_words + id_slots * 4) * 128;
  const size_t smem_max = (size_t)c->smem_optin - 1024;
  const bool smem_tables = table_bytes + 4 * priv_per_warp <= smem_max;
  const size_t avail = smem_max - (smem_tables ? table_bytes : 0);
  int warps = (int)(avail / priv_per_warp);
  if (warps > 16) warps = 16;
  if (const char* e = getenv("WHP_WARPS")) { int v = atoi(e); if (v >= 1 && v <= warps) warps = v; }
  if (warps < 1) return cudaErrorInvalidConfiguration;
  const int64_t resident_warps = (int64_t)c->num_sms * warps;
  // segments: few enough batches per segment for the counter planes, and ~4 tasks per warp
  int S = 1;
  while (S < 32 && ((nb_ub + S - 1) / S > 255 || n_cand * S < 4 * resident_warps * 32)) S <<= 1;
  if (const char* e = getenv("WHP_SEGMENTS")) {
    int v = atoi(e);
    if (v >= 1 && v <= 32 && (v & (v - 1)) == 0 && (nb_ub + v - 1) / v <= 255) S = v;
  }
  int log2S = 0;
  while ((1 << log2S) < S) ++log2S;
  int seg_planes = 1;  // planes of one segment's counters; one more per combine level
  while ((1ll << seg_planes) <= (nb_ub + S - 1) / S) ++seg_planes;
  const bool depot0_pl = c->g.depot_aisle == 0;
  const int kernel_planes = (depot0_pl && seg_planes <= 6) ? 6 : 8;  // the instantiation used
  const int planes_used = kernel_planes + log2S;
  // scratch (grow-only; reallocated when the shape changes)
  const int64_t plane_words = (int64_t)(kMaxPlanes + 5) * KW;
  if (c->fast_cap < n_cand || c->fast_pitch != bm_pitch || c->fast_plane_words < plane_words) {
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    cudaFree(c->d_bmask); cudaFree(c->d_cstream); cudaFree(c->d_nb); cudaFree(c->d_dist_scratch);
    cudaFree(c->d_planes);
    c->d_bmask = nullptr; c->d_cstream = nullptr; c->d_nb = nullptr; c->d_dist_scratch = nullptr;
    c->d_planes = nullptr;
    const int64_t cap = n_cand > c->fast_cap ? n_cand : c->fast_cap;
    const int64_t pw = plane_words > c->fast_plane_words ? plane_words : c->fast_plane_words;
    c->fast_cap = 0;
    if ((e = cudaMalloc(&c->d_bmask, 4 * (size_t)cap * bm_pitch)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_cstream, 2 * (size_t)cap * cs_pitch + 64)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_nb, 4 * (size_t)cap)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_dist_scratch, 8 * (size_t)cap)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_planes, 4 * (size_t)cap * pw)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(c->d_bmask, 0, 4 * (size_t)cap * bm_pitch, st)) != cudaSuccess) return e;
    c->fast_cap = cap; c->fast_pitch = bm_pitch; c->fast_plane_words = pw;
  }
  // K1
  {
    cudaError_t e = cudaMemsetAsync(c->d_task, 0, 2 * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    const size_t smem = (size_t)kRing * kBoundsThreads * 16 + 4 * (size_t)c->n_orders;
    cudaFuncSetAttribute(whp_bounds_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
    const unsigned blocks = (unsigned)((n_cand + kBoundsThreads - 1) / kBoundsThreads);
    whp_bounds_kernel<<<blocks, kBoundsThreads, smem, st>>>(
        c->d_order_fast, c->n_orders, c->C, d_perms, n_cand, c->d_bmask, bm_pitch, c->d_cstream,
        cs_pitch, c->d_nb, out.n_batches);
    c->launches += 1;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  // K2
  {
    sets_params P;
    P.S = S; P.log2S = 0; while ((1 << P.log2S) < S) ++P.log2S;
    P.aw_words = aw_words; P.ring_words = ring_words; P.id_slots = id_slots;
    P.bm_pitch = bm_pitch; P.cs_pitch = cs_pitch; P.n_items_pad = c->n_items_pad;
    P.n_tasks = (n_cand * S + 31) / 32;
    int64_t blocks = (P.n_tasks + warps - 1) / warps;
    if (blocks > c->num_sms) blocks = c->num_sms;
    const size_t smem = (smem_tables ? table_bytes : 0) + priv_per_warp * warps;
    const bool depot0 = c->g.depot_aisle == 0;
#define WHP_LAUNCH_SETS_PL(ST, D0, KWV, PLV)                                                     \
  do {                                                                                           \
    cudaFuncSetAttribute(whp_sets_kernel<ST, D0, KWV, PLV>,                                      \
                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);            \
    whp_sets_kernel<ST, D0, KWV, PLV><<<(unsigned)blocks, warps * 32, smem, st>>>(               \
        T, P, c->d_pick_fast, c->d_cstream, c->d_bmask, c->d_nb, n_cand, c->d_dist_scratch,      \
        c->d_planes, out.batch_hash, c->d_task);                                                 \
  } while (0)
#define WHP_LAUNCH_SETS(ST, D0, KWV)                                                             \
  do {                                                                                           \
    if (D0 && seg_planes <= 6) WHP_LAUNCH_SETS_PL(ST, D0, KWV, 6);                               \
    else WHP_LAUNCH_SETS_PL(ST, D0, KWV, 8);                                                     \
  } while (0)
#define WHP_LAUNCH_SETS_KW(ST, D0)                                                               \
  do {                                                                                           \
    if (KW == 1) WHP_LAUNCH_SETS(ST, D0, 1);                                                     \
    else if (KW == 2) WHP_LAUNCH_SETS(ST, D0, 2);                                                \
    else if (KW == 4) WHP_LAUNCH_SETS(ST, D0, 4);                                                \
    else if (KW == 7) WHP_LAUNCH_SETS(ST, D0, 7);                                                \
    else WHP_LAUNCH_SETS(ST, D0, 8);                                                             \
  } while (0)
    if (smem_tables && depot0) WHP_LAUNCH_SETS_KW(true, true);
    else if (smem_tables) WHP_LAUNCH_SETS_KW(true, false);
    else if (depot0) WHP_LAUNCH_SETS_KW(false, true);
    else WHP_LAUNCH_SETS_KW(false, false);
#undef WHP_LAUNCH_SETS_KW
#undef WHP_LAUNCH_SETS
#undef WHP_LAUNCH_SETS_PL
    c->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  // K3
  if (out.dist || out.penalty || out.obj || out.resp) {
    const unsigned blocks = (unsigned)((n_cand * 32 + 255) / 256);
    whp_finish_kernel<<<blocks, 256, 0, st>>>(T, n_cand, c->d_dist_scratch, c->d_planes, KW,
                                              planes_used, out.dist, out.penalty, out.obj,
                                              out.resp);
    c->launches += 1;
    return cudaGetLastError();
  }
  return cudaSuccess;
}
