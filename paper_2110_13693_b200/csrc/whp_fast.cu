// whp_fast.cu — the tuned candidate path: kernels with no cross-lane operation
// inside their inner loops.
//
//   K1 whp_bounds_kernel    one THREAD per plan runs the next-fit recurrence (D2) over its row of
//                           the permutation matrix, which arrives as 2-D TMA tiles (32 plans x 32
//                           positions, 128-byte swizzle, mbarrier pipeline). It writes (i) a
//                           bitmask of batch-start positions and (ii) the "cursor stream": for
//                           every position the 16-bit index of the order's first pick record, so
//                           K2 needs neither the permutation nor the order table (out through
//                           swizzled shared-memory tiles and TMA tile stores).
//      whp_segments_kernel  one warp per plan: batch count, first position of every segment.
//      whp_bop_kernel       optional batch_of_pos from the bitmask.
//   K2 whp_sets_kernel      one LANE per (plan, segment): a plan's batches are cut into S equal
//                           runs; a lane walks the picks of its run, one pick per branch-free
//                           step. Its occupancy sets are PRIVATE 32-bit shared-memory words laid
//                           out [word][lane] (bank = lane: never a bank conflict), addressed as
//                           base | offset. At the batch close: m = sum of popc, the words are
//                           cleared, S-shape length (D4) from m and the max pick record; the
//                           batch's class set is added into bit-sliced ("vertical") counters
//                           held in registers (D5). With S = 32 it also decodes r_k.
//   KL whp_legs_kernel      NEXT-2: K2's decomposition without the sets — a step adds the leg
//                           from the previous pick (D0's walking metric).
//   K3 whp_finish_kernel    one warp per plan: r_k, canonical fp64 penalty (D6), J, outputs.
#include <cuda.h>
#include <cudaTypedefs.h>

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

// Programmatic dependent launch (as in whp_swaps.cu): K2 may become resident — and stage its pick
// table — while the segments kernel drains; it passes dep_wait() before it reads anything K1 or
// the segments kernel wrote.
__device__ __forceinline__ void dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void dep_trigger() { asm volatile("griddepcontrol.launch_dependents;"); }

// ------------------------------------------------------------------------------------------ K1
// Next-fit batching (D2) is a sequential recurrence along the plan: one thread per plan, one
// warp per block. The plans of a warp are 32 consecutive rows of the permutation matrix, so one
// 2-D TMA tile load (tensor map over perms, box = 32 rows x 32 positions, 128-byte swizzle)
// brings one 32-position word of all 32 plans with a single instruction; kStages tiles are in flight
// per warp (an mbarrier per stage). The swizzle makes the lane-per-row 128-bit reads
// conflict-free. The loop is software-pipelined by hand — while the recurrence runs over word w,
// the order ids of word w+1 leave the tile and their order records are gathered from the table
// in shared memory — so that a lone warp per scheduler keeps issuing.
constexpr int kStages = 6;           // tiles (words) in flight per warp (seven are no faster alone
                                     // and leave four one-warp blocks 12 KB of an SM's shared memory:
                                     // with six, two blocks of another stream's kernel fit beside them)
constexpr int kStagesWide = 5;       // ... of the five-warp block (multi-wave launches, see bounds_shape)
constexpr int kTileBytes = 32 * 128; // 32 rows x 32 positions x 4 B

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// TMA bulk copy global -> shared, completion counted in bytes on the mbarrier
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// TMA 2-D tile store shared -> global (bulk async-group completion)
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* tm, int32_t x, int32_t y, uint32_t src) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
               ::"l"(tm), "r"(x), "r"(y), "r"(src) : "memory");
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
// TMA 2-D tile load: box at (x = first position, y = first plan) of the tensor map
__device__ __forceinline__ void tma_tile_2d(uint32_t dst, const CUtensorMap* tm, int32_t x, int32_t y,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(dst), "l"(tm), "r"(x), "r"(y), "r"(bar) : "memory");
}

// order records of the positions of a word (ids from the staged chunk, records from the order
// table in shared memory). FULL: all 32 positions, straight-line code; otherwise only the first
// n4 groups of four exist and the others get record 0 (q = 0: no effect on the recurrence).
// U16: the plans hold 16-bit order ids; a 128-byte tile row is then two words (64 positions) and
// `half` selects the word (chunks 4 half .. 4 half + 3, eight ids each).
template <bool FULL, bool U16>
__device__ __forceinline__ void gather_word(uint32_t (&r)[32], uint32_t row, uint32_t swz,
                                            uint32_t sorec0, int n4, int left = 32, int half = 0) {
  // row = address of this lane's 128-byte row of the tile; 16-byte chunk g lives at g ^ (lane & 7)
  if (U16) {
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      if (FULL || 2 * g < n4) {
        const int4 v = lds128(row + ((16 * (g + 4 * half)) ^ swz));
        const uint32_t w4[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          r[8 * g + 2 * j] = lds32(sorec0 + ((w4[j] << 2) & 0x3fffcu));
          r[8 * g + 2 * j + 1] = lds32(sorec0 + ((w4[j] >> 14) & 0x3fffcu));
        }
      } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) r[8 * g + j] = 0u;
      }
    }
  } else {
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      if (FULL || g < n4) {
        const int4 v = lds128(row + ((16 * g) ^ swz));
        r[4 * g + 0] = lds32(sorec0 + 4 * v.x); r[4 * g + 1] = lds32(sorec0 + 4 * v.y);
        r[4 * g + 2] = lds32(sorec0 + 4 * v.z); r[4 * g + 3] = lds32(sorec0 + 4 * v.w);
      } else {
        r[4 * g + 0] = 0u; r[4 * g + 1] = 0u; r[4 * g + 2] = 0u; r[4 * g + 3] = 0u;
      }
    }
  }
  if (!FULL) {  // a plan whose length is no multiple of 4: the tile is zero-filled past its end
#pragma unroll
    for (int i = 0; i < 32; ++i)
      if (i >= left) r[i] = 0u;
  }
}

// The next-fit recurrence over one word, on room = C - load:  room' = umin(room - q, C - q)
// (room < q wraps room - q above C - q: a new batch opens) — ONE dependent instruction per
// position (a fused add-min); everything else hangs off the chain: d = room - q is negative
// exactly when a batch opens, and a funnel shift collects the 32 sign bits, first position last. Writes the 16-bit cursors (bits 8..23 of the order records) of the first n4
// groups of four positions.
// TILE: the cursors go to this lane's 128-byte row of a shared-memory tile (two words per
// row, 16-byte chunk c at c ^ (lane & 7)) that a TMA tile store writes out; otherwise straight
// to global memory (tail words).
template <bool FULL, bool TILE>
__device__ __forceinline__ uint32_t recur_word(const uint32_t (&r)[32], uint32_t C, uint32_t& room,
                                               uint4* __restrict__ cs_out, uint32_t out_row,
                                               uint32_t swz, int half, int n4, bool write) {
  uint32_t rev = 0;
#pragma unroll
  for (int i = 0; i < 32; ++i) {
    uint32_t ri = r[i];
    // the records were gathered one phase ago: keep the scheduler from pulling their first
    // use up to the loads (it would stall on the shared-memory latency there)
    asm volatile("" : "+r"(ri));
    const uint32_t q = ri & WHP_Q_MASK;
    const uint32_t d = room - q;       // wraps (sign bit set) <=> room < q: a batch opens here
    rev = __funnelshift_l(d, rev, 1);  // (rev << 1) | (d >> 31)
    room = min(room + (0u - q), C - q);
  }
#pragma unroll
  for (int g2 = 0; g2 < 4; ++g2) {
    if (FULL || 2 * g2 < n4) {
      const uint32_t c0 = __byte_perm(r[8 * g2 + 0], r[8 * g2 + 1], 0x6521);
      const uint32_t c1 = __byte_perm(r[8 * g2 + 2], r[8 * g2 + 3], 0x6521);
      const uint32_t c2 = __byte_perm(r[8 * g2 + 4], r[8 * g2 + 5], 0x6521);
      const uint32_t c3 = __byte_perm(r[8 * g2 + 6], r[8 * g2 + 7], 0x6521);
      if (TILE) {
        asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(out_row + ((16 * (g2 + 4 * half)) ^ swz)),
                     "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
      } else if (write) {
        cs_out[g2] = make_uint4(c0, c1, c2, c3);
      }
    }
  }
  return __brev(rev);
}

// kWarps: warps per block, they share the order table (a warp = 32 plans). U16: the plan matrix
// holds 16-bit order ids (whp_eval_candidates_host16): a tile is then 32 plans x 64 positions.
// kSt: tiles in flight per warp.
template <int kWarps, bool U16, int kSt>
__global__ void __launch_bounds__(32 * kWarps)
whp_bounds_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_cs,
                  const uint32_t* __restrict__ order_fast,
                  int32_t n_orders, int32_t C, int64_t n_cand, uint32_t* __restrict__ bmask,
                  int32_t bm_pitch, uint16_t* __restrict__ cstream, int32_t cs_pitch) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  // per warp: [tiles: kSt x 4 KB, 1 KB aligned (swizzle)][cursor tiles: 2 x 4 KB]; then
  // the order table shared by the block's warps and the mbarriers (kSt per warp + 1)
  const int nw = (n_orders + 31) >> 5;
  const int lane = threadIdx.x & 31, wq = threadIdx.x >> 5;
  const uint32_t area = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t tiles = area + wq * (kSt + 2) * kTileBytes;
  const uint32_t otiles = tiles + kSt * kTileBytes;  // 32 rows x 64 cursors, two of them
  const uint32_t sorec0 = area + kWarps * (kSt + 2) * kTileBytes;
  const uint32_t bar_table = sorec0 + 4u * (uint32_t)((n_orders + 3) & ~3);
  const uint32_t bars = bar_table + 8 + 8 * kSt * wq;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kSt * kWarps + 1; ++s) mbar_init(bar_table + 8 * s, 1);
  }
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();
  const int64_t row0 = ((int64_t)blockIdx.x * kWarps + wq) * 32;  // first plan of this warp
  const int nt = U16 ? (nw + 1) >> 1 : nw;  // tiles of a plan
  auto issue = [&](int t) {  // one lane: tile t into stage t mod kSt
    const uint32_t bar = bars + 8 * (t % kSt);
    mbar_expect_tx(bar, kTileBytes);
    tma_tile_2d(tiles + (t % kSt) * kTileBytes, &tmap, (U16 ? 64 : 32) * t, (int32_t)row0, bar);
  };
  if (threadIdx.x == 0) {  // the order table: one bulk copy (n_orders is a multiple of 4)
    const uint32_t table_bytes = 4u * (uint32_t)((n_orders + 3) & ~3);  // the table is padded
    mbar_expect_tx(bar_table, table_bytes);
    bulk_g2s(sorec0, order_fast, table_bytes, bar_table);
  }
  if (lane == 0)
    for (int t = 0; t < kSt && t < nt; ++t) issue(t);
  const int64_t c = row0 + lane;
  const bool have = c < n_cand;  // rows past the end arrive zero-filled: order 0, never written
  uint32_t* __restrict__ bm = bmask + (have ? c : 0) * bm_pitch;
  uint4* __restrict__ cs = reinterpret_cast<uint4*>(cstream + (have ? c : 0) * cs_pitch);
  const uint32_t rowoff = lane * 128, swz = (lane & 7) << 4;
  auto tile_of = [&](int w) { return U16 ? w >> 1 : w; };
  auto tile_row = [&](int w) { return tiles + (tile_of(w) % kSt) * kTileBytes + rowoff; };
  auto wait_word = [&](int w) {
    mbar_wait(bars + 8 * (tile_of(w) % kSt), (tile_of(w) / kSt) & 1);
  };
  auto refill = [&](int w) {  // word w is consumed by every lane: its stage takes the next tile
    // (the tile was only READ, and every value read has been used: no proxy fence is needed
    // before the async proxy overwrites it)
    if (U16 && !(w & 1)) return;  // the tile's second word is still to come
    __syncwarp();
    if (lane == 0 && tile_of(w) + kSt < nt) issue(tile_of(w) + kSt);
  };
  uint32_t room = (uint32_t)C;
  uint32_t ra[32], rb[32];
  mbar_wait(bar_table, 0);
  wait_word(0);
  const int n_full = n_orders >> 5;            // words with all 32 positions
  // pairs of words (2k, 2k+1) whose successor 2k+2 is full too: the straight-line path
  const int KF = n_full > 0 ? (n_full - 1) >> 1 : 0;
  if (n_full > 0) gather_word<true, U16>(ra, tile_row(0), swz, sorec0, 8, 32, 0);
#pragma unroll 1
  for (int k = 0; k < KF; ++k) {
    const int w = 2 * k;
    const uint32_t otile = otiles + (k & 1) * kTileBytes;
    // the tile store issued two iterations ago must have read this cursor tile
    if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
    __syncwarp();
    // word w runs its recurrence while word w+1 is gathered
    wait_word(w + 1);
    gather_word<true, U16>(rb, tile_row(w + 1), swz, sorec0, 8, 32, 1);
    uint32_t bits = recur_word<true, true>(ra, (uint32_t)C, room, nullptr, otile + rowoff, swz, 0, 8, have);
    if (k == 0) bits |= 1u;  // batch 0 starts at position 0
    const uint32_t bits_even = bits;
    refill(w);
    // word w+1 runs its recurrence while word w+2 is gathered
    wait_word(w + 2);
    gather_word<true, U16>(ra, tile_row(w + 2), swz, sorec0, 8, 32, 0);
    bits = recur_word<true, true>(rb, (uint32_t)C, room, nullptr, otile + rowoff, swz, 1, 8, have);
    if (have) *reinterpret_cast<uint2*>(bm + w) = make_uint2(bits_even, bits);
    refill(w + 1);
    // the 64 cursors of words w, w+1 of all 32 plans: one tile store (rows past n_cand clipped)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if (lane == 0) tma_store_2d(&tmap_cs, 32 * w, (int32_t)row0, otile);
  }
  // the last (at most three) words, the final one possibly partial; word 2*KF is in ra if full
#pragma unroll 1
  for (int w = 2 * KF; w < nw; ++w) {
    const int left = n_orders - 32 * w;
    const int n4 = min(8, (left + 3) >> 2);
    if (w > 2 * KF || n_full == 0) {
      wait_word(w);
      gather_word<false, U16>(ra, tile_row(w), swz, sorec0, n4, left, w & 1);
    }
    uint32_t bits = recur_word<false, false>(ra, (uint32_t)C, room, cs + 4 * w, 0u, 0u, 0, n4, have);
    if (w == 0) bits |= 1u;
    if (left < 32) bits |= 1u << left;    // end sentinel in a partial last word
    if (have) bm[w] = bits;
  }
  if (have && (n_orders & 31) == 0) bm[nw] = 1u;  // end sentinel in a word of its own
  if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");  // tiles still being read
}

// The register path of whp_segments_kernel: lane l owns the 4*W4 consecutive mask words from
// 4*W4*l on (16-byte loads), so one warp scan over the lanes' totals ranks every word; a segment
// then finds its lane by a shuffle binary search, the word inside that lane from the lane's
// packed per-word counts, and the bit by clearing the lower ones.
template <int W4>
__device__ __forceinline__ void segments_in_registers(
    const uint32_t* __restrict__ bm, int32_t bm_pitch, int32_t n_orders, int nw, int lane, int32_t S,
    int32_t log2S, int64_t c, int32_t* __restrict__ nb_scratch, int32_t* __restrict__ n_batches_out,
    int32_t* __restrict__ segstart, int32_t ss_pitch) {
  constexpr int W = 4 * W4;
  uint32_t x[W], pk[W4];
  const int w0 = lane * W;
  const int ws = n_orders >> 5;  // the word that also holds the end sentinel (n_orders % 32 != 0)
  int tot = 0;
#pragma unroll
  for (int i4 = 0; i4 < W4; ++i4) {
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (w0 + 4 * i4 < bm_pitch) v = __ldg(reinterpret_cast<const uint4*>(bm + w0 + 4 * i4));
    x[4 * i4 + 0] = v.x; x[4 * i4 + 1] = v.y; x[4 * i4 + 2] = v.z; x[4 * i4 + 3] = v.w;
    pk[i4] = 0u;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int w = w0 + 4 * i4 + k;
      uint32_t xi = x[4 * i4 + k];
      if (w >= nw) xi = 0u;
      else if (w == ws) xi &= (1u << (n_orders & 31)) - 1u;  // drop the end sentinel
      x[4 * i4 + k] = xi;
      const int pc = __popc(xi);
      pk[i4] |= (uint32_t)pc << (8 * k);
      tot += pc;
    }
  }
  int incl = tot;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int y = __shfl_up_sync(WHP_FULL, incl, d);
    if (lane >= d) incl += y;
  }
  const int nb = __shfl_sync(WHP_FULL, incl, 31);
  if (lane == 0) {
    nb_scratch[c] = nb;
    if (n_batches_out) n_batches_out[c] = nb;
  }
  const int target = (int)(((int64_t)lane * nb) >> log2S);  // lane = segment
  int lo = 0, hi = 31;  // smallest lane whose inclusive count exceeds the target
#pragma unroll
  for (int it = 0; it < 5; ++it) {
    const int mid = (lo + hi) >> 1;
    const int im = __shfl_sync(WHP_FULL, incl, mid);
    if (im > target) hi = mid; else lo = mid + 1;
  }
  int r = target - __shfl_sync(WHP_FULL, incl - tot, lo);  // rank inside that lane's words
  int j = -1;
#pragma unroll
  for (int i4 = 0; i4 < W4; ++i4) {
    const uint32_t p = __shfl_sync(WHP_FULL, pk[i4], lo);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int pc = (int)((p >> (8 * k)) & 0xffu);
      if (j < 0) {
        if (r < pc) j = 4 * i4 + k; else r -= pc;
      }
    }
  }
  uint32_t t = 0u;
#pragma unroll
  for (int i = 0; i < W; ++i) {
    const uint32_t xi = __shfl_sync(WHP_FULL, x[i], lo);
    if (i == j) t = xi;
  }
  if (lane < S && j >= 0) {
    for (; r > 0; --r) t &= t - 1;
    segstart[c * ss_pitch + lane] = 32 * (lo * W + j) + __ffs(t) - 1;
  }
}

// One warp per plan: number of batches, and the first position of every segment (segment s
// starts with batch floor(s * nb / S)).
__global__ void __launch_bounds__(256)
whp_segments_kernel(const uint32_t* __restrict__ bmask, int32_t bm_pitch, int32_t n_orders,
                    int64_t n_cand, int32_t S, int32_t log2S, int32_t* __restrict__ nb_scratch,
                    int32_t* __restrict__ n_batches_out, int32_t* __restrict__ segstart,
                    int32_t ss_pitch) {
  dep_trigger();
  const int lane = threadIdx.x & 31;
  const int64_t c = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (c >= n_cand) return;
  const int nw = (n_orders + 31) >> 5;
  const uint32_t* __restrict__ bm = bmask + c * bm_pitch;
  auto word_at = [&](int w) -> uint32_t {
    if (w >= nw) return 0u;
    uint32_t x = __ldg(bm + w);
    if (w == (n_orders >> 5)) x &= (1u << (n_orders & 31)) - 1u;  // drop the end sentinel
    return x;
  };
  // masks of up to 640 words: lane l keeps words 4*W4*l .. 4*W4*(l+1)-1 in registers
  switch ((nw + 127) >> 7) {
    case 1: segments_in_registers<1>(bm, bm_pitch, n_orders, nw, lane, S, log2S, c, nb_scratch, n_batches_out, segstart, ss_pitch); return;
    case 2: segments_in_registers<2>(bm, bm_pitch, n_orders, nw, lane, S, log2S, c, nb_scratch, n_batches_out, segstart, ss_pitch); return;
    case 3: segments_in_registers<3>(bm, bm_pitch, n_orders, nw, lane, S, log2S, c, nb_scratch, n_batches_out, segstart, ss_pitch); return;
    case 4: segments_in_registers<4>(bm, bm_pitch, n_orders, nw, lane, S, log2S, c, nb_scratch, n_batches_out, segstart, ss_pitch); return;
    case 5: segments_in_registers<5>(bm, bm_pitch, n_orders, nw, lane, S, log2S, c, nb_scratch, n_batches_out, segstart, ss_pitch); return;
    default: break;
  }
  int nb = 0;
  for (int w0 = 0; w0 < nw; w0 += 32) nb += __reduce_add_sync(WHP_FULL, __popc(word_at(w0 + lane)));
  if (lane == 0) {
    nb_scratch[c] = nb;
    if (n_batches_out) n_batches_out[c] = nb;
  }
  const int target = (int)(((int64_t)lane * nb) >> log2S);  // lane = segment
  int base = 0, found = 0;
  for (int w0 = 0; w0 < nw; w0 += 32) {
    const uint32_t x = word_at(w0 + lane);
    const int pc = __popc(x);
    int incl = pc;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int y = __shfl_up_sync(WHP_FULL, incl, d);
      if (lane >= d) incl += y;
    }
    const int total = __shfl_sync(WHP_FULL, incl, 31);
    // smallest j with base + incl_j > target
    int lo = 0, hi = 31;
#pragma unroll
    for (int it = 0; it < 5; ++it) {
      const int mid = (lo + hi) >> 1;
      const int im = __shfl_sync(WHP_FULL, incl, mid);
      if (base + im > target) hi = mid; else lo = mid + 1;
    }
    const uint32_t xj = __shfl_sync(WHP_FULL, x, lo);
    const int ej = __shfl_sync(WHP_FULL, incl - pc, lo);
    if (!found && lane < S && target >= base && target < base + total) {
      uint32_t t = xj;
      for (int r = target - base - ej; r > 0; --r) t &= t - 1;
      segstart[c * ss_pitch + lane] = 32 * (w0 + lo) + __ffs(t) - 1;
      found = 1;
    }
    base += total;
  }
}

// batch_of_pos (D2, optional output) from the boundary mask: one warp per plan, a running batch
// count over the words, lane i of word w writes position 32w + i (coalesced).
__global__ void __launch_bounds__(256)
whp_bop_kernel(const uint32_t* __restrict__ bmask, int32_t bm_pitch, int32_t n_orders,
               int64_t n_cand, int32_t* __restrict__ batch_of_pos) {
  const int lane = threadIdx.x & 31;
  const int64_t c = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (c >= n_cand) return;
  const int nw = (n_orders + 31) >> 5;
  const uint32_t* __restrict__ bm = bmask + c * bm_pitch;
  int32_t* __restrict__ row = batch_of_pos + c * n_orders;
  int32_t before = 0;  // batches that start before the current word
  for (int w = 0; w < nw; ++w) {
    uint32_t x = __ldg(bm + w);
    if (w == (n_orders >> 5)) x &= (1u << (n_orders & 31)) - 1u;  // drop the end sentinel
    const int32_t p = 32 * w + lane;
    if (p < n_orders) row[p] = before + __popc(x & (WHP_FULL >> (31 - lane))) - 1;
    before += __popc(x);
  }
}

// ------------------------------------------------------------------------------------------ K2
// vertical counter bit planes: at most 8 per segment (up to 255 batches) + 5 combine levels
constexpr int kPlaneRow = 16;  // words per class word in a plan's counter row: 13 planes, or
                               // (S = 32) the 32 decoded 16-bit counts

struct sets_params {
  int S;           // segments per candidate (power of two <= 32)
  int log2S;
  int aw_words;    // 32-aisle occupancy words per lane = ceil(NA/32)
  int awp;         // aw_words rounded up to a power of two: a warp's aisle words are awp*128 B
  int kwp;         // the same for the KW class words
  int ring_mask;   // bytes of the per-lane cursor ring - 1 (ring = 8 or 16 chunks of 16 B)
  int bm_pitch, cs_pitch, ss_pitch;
  int n_items_pad;
  int fits32;      // every per-batch length fits 31 bits
  int64_t n_tasks;  // warp tasks = ceil(n_cand*S/32)
};

__device__ __forceinline__ uint32_t lds16(uint32_t a) {
  uint32_t v; asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(a)); return v;
}

// One step's cursor transition for pick tables in shared memory, written in PTX so that the bit
// test lands in a predicate and every update is a single predicated instruction:
//   last = rec & LAST;  more = last && v != v_end;
//   cur  = more ? pb + 8 * n_c16 : (last ? cur : cur + 4);
//   if (more) { v += 2;  n_c16 = ld.shared.u16 [ringbase + (v & ring_mask)]; }
__device__ __forceinline__ void step_cursor(uint32_t rec, uint32_t& cur, uint32_t& v, uint32_t v_end,
                                            uint32_t& n_c16, uint32_t pb, uint32_t ringbase,
                                            uint32_t ring_mask) {
  asm volatile(
      "{\n"
      ".reg .pred pl, pm;\n"
      ".reg .b32 t;\n"
      "and.b32 t, %3, 0x20;\n"
      "setp.ne.u32 pl, t, 0;\n"
      "setp.ne.and.u32 pm, %1, %4, pl;\n"
      "@!pl add.u32 %0, %0, 4;\n"
      "@pm mad.lo.u32 %0, %2, 8, %5;\n"
      "@pm add.u32 %1, %1, 2;\n"
      "and.b32 t, %1, %7;\n"
      "add.u32 t, t, %6;\n"
      "@pm ld.shared.u16 %2, [t];\n"
      "}\n"
      : "+r"(cur), "+r"(v), "+r"(n_c16)
      : "r"(rec), "r"(v_end), "r"(pb), "r"(ringbase), "r"(ring_mask));
}

// if (p) {a, b} = the aligned record pair at ptr (ld.global.nc.v2) — predicated, never a branch.
// Pick tables that do not fit shared memory are gathered through L1 / L2, where a warp-wide
// gather costs one tag look-up per lane (the L1TEX unit is what saturates: 91 % at stress scale):
// every order starts at an even index, so one 8-byte load serves two consecutive steps.
__device__ __forceinline__ void ldg_pair_if(uint32_t& a, uint32_t& b, const uint32_t* ptr, bool p) {
  asm volatile("{ .reg .pred pq; setp.ne.u32 pq, %3, 0; @pq ld.global.nc.v2.u32 {%0, %1}, [%2]; }"
               : "+r"(a), "+r"(b) : "l"(ptr), "r"((uint32_t)p));
}

// if (p) v = ld.shared.u16 [a] — predicated, never a branch; idle lanes cost no bank cycle
__device__ __forceinline__ void lds16_if(uint32_t& v, uint32_t a, bool p) {
  asm volatile("{ .reg .pred pq; setp.ne.u32 pq, %2, 0; @pq ld.shared.u16 %0, [%1]; }"
               : "+r"(v) : "r"(a), "r"((uint32_t)p));
}

// SMEM_TABLES false: the pick table does not fit shared memory and is gathered through L1 / L2
// (the shared memory the private state leaves free is L1: 32 warps instead of 24 leave 10 KB of it
// and the stress evaluation goes from 10.6 to 17.5 ms, the L1 hit rate from 52 % to 2 %).
template <bool SMEM_TABLES, bool DEPOT0, int KW, int kPlanes>
__global__ void __launch_bounds__(KW * kPlanes <= 42 ? 768 : 512, 1)  // counter registers: KW x planes
whp_sets_kernel(const whp_tables T, const sets_params P, const uint32_t* __restrict__ pick_fast,
                const uint16_t* __restrict__ cstream, const uint32_t* __restrict__ bmask,
                const int32_t* __restrict__ nb_scratch, const int32_t* __restrict__ segstart,
                int64_t n_cand, int64_t* __restrict__ dist_scratch,
                uint32_t* __restrict__ planes_out, uint64_t* __restrict__ hash_out,
                unsigned long long* __restrict__ task_counter, int64_t* __restrict__ o_dist,
                double* __restrict__ o_pen, double* __restrict__ o_obj, int32_t* __restrict__ o_resp) {
  extern __shared__ __align__(16) uint32_t smem[];
  // layout: [pick table n_items_pad] (if staged) [per-warp private words]
  uint32_t* priv = smem;
  uint32_t pick_base = 0;
  if (SMEM_TABLES) {
    for (int i = threadIdx.x; i < P.n_items_pad; i += blockDim.x) smem[i] = __ldg(pick_fast + i);
    pick_base = smem_u32(smem);
    priv = smem + ((P.n_items_pad + 31) & ~31);
    __syncthreads();
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int nwarps = blockDim.x >> 5;
  // private state of a lane: aw_words aisle words and KW class words laid out [word][lane]
  // (bank = lane), a warp's words aligned to their (power-of-two) size so that a word's
  // address is base | offset; then the lane's cursor ring, lane-major, stride ring + 16 bytes
  const int ring_stride = P.ring_mask + 1 + 16;
  const uint32_t a_area = (smem_u32(priv) + P.awp * 128 - 1) & ~(uint32_t)(P.awp * 128 - 1);
  const uint32_t c_area = a_area + nwarps * P.awp * 128;  // awp >= kwp: aligned as well
  const uint32_t abase = a_area + warp * P.awp * 128 + lane * 4;
  const uint32_t cbase = c_area + warp * P.kwp * 128 + lane * 4;
  const uint32_t ringbase = c_area + nwarps * P.kwp * 128 + (warp * 32 + lane) * ring_stride;
  const uint32_t amask = (uint32_t)(P.awp - 1) << 7;
  uint32_t pb;  // pinned in a register (the shared-window conversion is otherwise re-derived)
  asm volatile("mov.u32 %0, %1;" : "=r"(pb) : "r"(pick_base));
  const int chunks = (P.ring_mask + 1) >> 4;
  const int Cmax = T.C;
  const int64_t A = T.g.aisle_len;
  const int64_t P2 = 2 * (int64_t)T.g.aisle_spacing;
  const int n8 = P.cs_pitch >> 3;  // 16-byte chunks per cursor-stream row
  for (int w = 0; w < P.aw_words; ++w) sts32(abase + w * 128, 0u);
  for (int w = 0; w < KW; ++w) sts32(cbase + w * 128, 0u);
  dep_wait();  // everything above reads only the pick table: it overlaps the segments kernel

  __shared__ unsigned long long s_task[32];
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
    int b_lo = 0, nbseg = 0;
    if (have) {
      const int nb = __ldg(nb_scratch + cand);
      b_lo = (int)((int64_t)seg * nb >> P.log2S);
      nbseg = (int)((int64_t)(seg + 1) * nb >> P.log2S) - b_lo;
    }
    const int nbmax = __reduce_max_sync(WHP_FULL, nbseg);
    uint32_t pl[kPlanes][KW];
#pragma unroll
    for (int p = 0; p < kPlanes; ++p)
#pragma unroll
      for (int w = 0; w < KW; ++w) pl[p][w] = 0;

    // ---- first batch of the segment: its start position comes from K1
    const uint32_t* __restrict__ bm = bmask + cand * P.bm_pitch;
    int p = __ldg(segstart + cand * P.ss_pitch + seg);
    int wi = p >> 5;
    uint32_t bw = __ldg(bm + wi) & (WHP_FULL << (p & 31));
    uint32_t bw_next = __ldg(bm + min(wi + 1, P.bm_pitch - 1));

    // ---- cursor stream of this lane through its private cp.async ring: chunk c (cursors of
    // positions 8c..8c+7) lives at ring offset (16 c) mod ring
    const uint4* __restrict__ cs = reinterpret_cast<const uint4*>(cstream + cand * P.cs_pitch);
    // the last chunk this lane reads: the one that holds the first position of the next segment
    // (a third of the ring traffic used to be chunks fetched past the end of the lane's run)
    int c_last;
    {
      const int p_next = __shfl_down_sync(WHP_FULL, p, 1);
      c_last = min((seg == P.S - 1 || lane == 31 ? T.n_orders : p_next) >> 3, n8 - 1);
    }
    int lo_prev;  // first chunk that was resident when the newest refill group was issued
    {
      const int c0 = p >> 3;
      for (int k = 0; k < chunks; ++k)
        if (c0 + k <= c_last) cp_async16(ringbase + (((c0 + k) << 4) & P.ring_mask), cs + c0 + k);
      cp_async_commit();
      lo_prev = c0 - chunks;
    }

    int64_t D = 0;
    uint64_t hash = 0;
    for (int j = 0; j < nbmax; ++j) {
      int left = 0;  // orders of batch j
      const int p0 = p;
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
      // the newest refill group brought chunks lo_prev+chunks ..; everything older has landed
      // after wait<1>. The batch reads cursors of positions p0 .. p (one ahead).
      if (live && (p >> 3) >= lo_prev + chunks) cp_async_wait<0>(); else cp_async_wait<1>();
      uint32_t v = live ? 2u * (uint32_t)p0 : 0u;          // 2 x position of the next order
      const uint32_t v_end = live ? 2u * (uint32_t)p : 0u;
      uint32_t cur;
      if (live) {
        const uint32_t c16 = lds16(ringbase + (v & P.ring_mask));
        cur = SMEM_TABLES ? pb + 8 * c16 : 2 * c16;
        v += 2;
      } else {
        cur = SMEM_TABLES ? pb : 0u;
      }
      uint32_t n_c16 = lds16(ringbase + (v & P.ring_mask));
      uint32_t pair_lo = 0, pair_hi = 0;  // !SMEM_TABLES: the aligned record pair that holds cur
      if (!SMEM_TABLES) ldg_pair_if(pair_lo, pair_hi, pick_fast + cur, true);  // cur is even here
      uint32_t rec = SMEM_TABLES ? lds32(cur) : pair_lo;
      uint32_t kmax = 0, kmin = 0xffffffffu;
      uint32_t cset = 0;  // KW == 1: class set of the batch
      int m = 0;          // distinct aisles of the batch, counted as they arrive
      // Branch-free step: every lane runs Cmax steps. A lane that has finished its batch stays
      // on the batch's final pick and re-inserts it (set inserts and max are idempotent); a
      // lane without a batch walks to the end of order 0 and stays there — its sets are
      // discarded at the close below.
#pragma unroll 2
      for (int t = 0; t < Cmax; ++t) {
        // cursor of the next step's pick: next record, the next order's first pick, or stay —
        // all by selects and one predicated load
        if (SMEM_TABLES) {
          step_cursor(rec, cur, v, v_end, n_c16, pb, ringbase, (uint32_t)P.ring_mask);
        } else {
          const uint32_t first_of_next = 2 * n_c16;
          const bool last = (int32_t)(rec << 26) < 0;  // WHP_FAST_LAST (bit 5) into the sign bit
          const bool more = last && (v != v_end);
          uint32_t nxt = last ? cur : cur + 1u;
          nxt = more ? first_of_next : nxt;
          v = more ? v + 2 : v;
          lds16_if(n_c16, ringbase + (v & P.ring_mask), more);  // the look-ahead cursor
          // a new pair is needed exactly when the cursor moved on to an even index (the next
          // pair of this order, or the first pick of the next order). Measured and not kept:
          // fetching the next order's first pair one order ahead (12.9 ms against 12.2 ms for
          // the 65,536 stress plans: the extra loads cost more than the hidden latency saves)
          ldg_pair_if(pair_lo, pair_hi, pick_fast + nxt, (nxt != cur) && !(nxt & 1u));
          cur = nxt;
        }
        const uint32_t rec_next = SMEM_TABLES ? lds32(cur) : ((cur & 1u) ? pair_hi : pair_lo);
        // ---- this step's pick
        kmax = max(kmax, rec);
        if (!DEPOT0) kmin = min(kmin, rec);
        const uint32_t aaddr = abase | ((rec >> 20) & amask);
        if (KW == 1) {  // up to 32 classes: the batch's class set is one register
          const uint32_t aw = lds32(aaddr), an = aw | one_shl_wrap(rec >> 22);
          m += (an != aw) ? 1 : 0;
          sts32(aaddr, an);
          cset |= one_shl_wrap(rec);
        } else {
          // the aisle word and the class word are different words: both loads go out before
          // either store, so a step waits for one shared-memory round trip instead of two
          const uint32_t caddr = cbase | (rec & 0x380u);
          const uint32_t aw = lds32(aaddr), cw = lds32(caddr);
          const uint32_t an = aw | one_shl_wrap(rec >> 22);
          m += (an != aw) ? 1 : 0;
          sts32(aaddr, an);
          sts32(caddr, cw | one_shl_wrap(rec));
        }
        rec = rec_next;
      }
      {  // refill the slots of the chunks this batch finished; waited for two batches later
        const int nf = live ? (p >> 3) - (p0 >> 3) : 0;
        const int nfmax = __reduce_max_sync(WHP_FULL, nf);
        for (int i = 0; i < nfmax; ++i) {
          const int c = (p0 >> 3) + i;
          if (i < nf && c + chunks <= c_last) cp_async16(ringbase + ((c << 4) & P.ring_mask), cs + c + chunks);
        }
        cp_async_commit();
        if (live) lo_prev = p0 >> 3;
      }
      // ---- close the batch: m = distinct aisles, D4; the sets are emptied for the next batch
#pragma unroll 4
      for (int w = 0; w < P.aw_words; ++w) sts32(abase + w * 128, 0u);
      if (live) {
        const uint32_t a_max = WHP_FAST_AISLE(kmax);
        const uint32_t slot1 = WHP_FAST_SLOT1(kmax);
        if (DEPOT0 && P.fits32) {
          const uint32_t d2 = 2u * slot1 * (uint32_t)T.g.slot_pitch;
          D += (uint32_t)P2 * a_max + (uint32_t)m * (uint32_t)A + ((m & 1) ? d2 - (uint32_t)A : 0u);
        } else {
          const int64_t d_last = (int64_t)slot1 * T.g.slot_pitch;
          int64_t H;
          if (DEPOT0) {
            H = P2 * (int64_t)a_max;
          } else {
            const int64_t a_min = WHP_FAST_AISLE(kmin), a0 = T.g.depot_aisle;
            H = (int64_t)T.g.aisle_spacing *
                (llabs(a0 - a_min) + ((int64_t)a_max - a_min) + llabs((int64_t)a_max - a0));
          }
          D += H + ((m & 1) ? (int64_t)(m - 1) * A + 2 * d_last : (int64_t)m * A);
        }
      }
      // the batch's class set goes into the vertical counters (D5)
#pragma unroll
      for (int w = 0; w < KW; ++w) {
        // lanes without a batch j ran the steps on a dummy pick: their set is discarded
        uint32_t carry;
        if (KW == 1) {
          carry = cset;
        } else {
          carry = lds32(cbase + w * 128);
          sts32(cbase + w * 128, 0u);
        }
        if (!live) carry = 0u;
#pragma unroll
        for (int pp = 0; pp < kPlanes; ++pp) {
          const uint32_t t2 = pl[pp][w] & carry;
          pl[pp][w] ^= carry;
          carry = t2;
        }
      }
    }
    cp_async_wait<0>();  // nothing of this task may still land in the ring
    // ---- combine the S segment lanes of each candidate (D, hash); write the counters
#pragma unroll
    for (int o = 1; o < 32; o <<= 1)
      if (o < P.S) {
        D += __shfl_xor_sync(WHP_FULL, D, o);
        hash += __shfl_xor_sync(WHP_FULL, hash, o);
      }
    const bool fused = P.S == 32;  // the warp is one plan: it finishes D6 itself (no K3)
    if (have && seg == 0) {
      if (!fused) dist_scratch[cand] = D;
      if (hash_out) hash_out[cand] = hash;
    }
    double phi = 0.0;
    // bit-sliced addition of the S lanes' vertical counters (one more plane per level)
    {
      uint32_t* __restrict__ po = planes_out + cand * (kPlaneRow * KW);
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
        if (fused) {
          // every lane holds the plan's counters: lane l decodes r_k of class 32w + l and adds
          // its term — ascending w, lane = k mod 32: the canonical accumulation of D6
          uint32_t r = 0;
#pragma unroll
          for (int pp = 0; pp < kPlanes + 5; ++pp) r |= ((a[pp] >> lane) & 1u) << pp;
          const int k = 32 * w + lane;
          if (k < T.K) {
            if (o_resp && have) o_resp[cand * T.K + k] = (int32_t)r;
            const double c = __dsub_rn(__ldg(T.tvw + k), (double)r);
            const double u = __dmul_rn(__ldg(T.tvw + 2 * T.K + k), c);
            phi = __dadd_rn(phi, __dadd_rn(__dmul_rn(__ldg(T.tvw + T.K + k), c), __dmul_rn(u, u)));
          }
        } else if (have && seg == 0) {
#pragma unroll
          for (int pp = 0; pp < kPlanes + 5; ++pp)
            if (pp < kPlanes + P.log2S) po[pp * KW + w] = a[pp];
        }
      }
    }
    if (fused) {
#pragma unroll
      for (int off = 16; off >= 1; off >>= 1) phi = __dadd_rn(phi, __shfl_xor_sync(WHP_FULL, phi, off));
      if (have && lane == 0) {
        if (o_dist) o_dist[cand] = D;
        if (o_pen) o_pen[cand] = phi;
        if (o_obj) o_obj[cand] = __dadd_rn((double)D, phi);
      }
    }
    __syncwarp();
  }
}

// ------------------------------------------------------------------------------------------ K2'
// K2 for pick tables that do not fit shared memory (stress scale: 305 KB) and are gathered
// through L1 / L2. The pair-load variant of whp_sets_kernel pays an L2 round trip per warp step
// of ONE pick: the address of a lane's next load depends on the last-pick flag of the record it
// is consuming, and with 32 lanes some lane needs a new pair at practically every step. Here the
// table is the four-aligned layout (whp_internal.cuh: every order starts at a multiple of four
// records and is padded to a multiple of four with copies of its last record — set inserts and
// max are idempotent) and a step is one 16-byte load = four picks, so a batch takes as many
// round trips as its longest lane has fours (~20 instead of C = 40 at stress scale) and the four
// inserts of a step cover the latency of the next load. The last record of an order's last four
// carries WHP_FAST_LAST4; a lane whose batch is exhausted keeps re-inserting its last four. The
// step loop ends when no lane of the warp has a four left.
__device__ __forceinline__ void lds64(uint32_t& lo, uint32_t& hi, uint32_t a) {
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(lo), "=r"(hi) : "r"(a));
}
__device__ __forceinline__ void lds64_if(uint32_t& lo, uint32_t& hi, uint32_t a, bool p) {
  asm volatile("{ .reg .pred pq; setp.ne.u32 pq, %3, 0; @pq ld.shared.v2.u32 {%0, %1}, [%2]; }"
               : "+r"(lo), "+r"(hi) : "r"(a), "r"((uint32_t)p));
}
__device__ __forceinline__ void ldg_four_if(uint4& q, const uint32_t* ptr, bool p) {
  asm volatile("{ .reg .pred pq; setp.ne.u32 pq, %5, 0; @pq ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4]; }"
               : "+r"(q.x), "+r"(q.y), "+r"(q.z), "+r"(q.w) : "l"(ptr), "r"((uint32_t)p));
}

template <bool DEPOT0, int KW, int kPlanes>
__global__ void __launch_bounds__(KW * kPlanes <= 16 ? 768 : 512, 1)  // the four records of a step + KW x planes counters
whp_sets4_kernel(const whp_tables T, const sets_params P, const uint32_t* __restrict__ pick_f4,
                const uint16_t* __restrict__ cstream, const uint32_t* __restrict__ bmask,
                const int32_t* __restrict__ nb_scratch, const int32_t* __restrict__ segstart,
                int64_t n_cand, int64_t* __restrict__ dist_scratch,
                uint32_t* __restrict__ planes_out, uint64_t* __restrict__ hash_out,
                unsigned long long* __restrict__ task_counter, int64_t* __restrict__ o_dist,
                double* __restrict__ o_pen, double* __restrict__ o_obj, int32_t* __restrict__ o_resp) {
  extern __shared__ __align__(16) uint32_t smem[];
  uint32_t* priv = smem;  // layout: [per-warp private words]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int nwarps = blockDim.x >> 5;
  // private state of a lane: aw_words aisle words and KW class words laid out [word][lane]
  // (bank = lane), a warp's words aligned to their (power-of-two) size so that a word's
  // address is base | offset; then the lane's cursor ring, lane-major, stride ring + 16 bytes
  const int ring_stride = P.ring_mask + 1 + 16;
  const uint32_t a_area = (smem_u32(priv) + P.awp * 128 - 1) & ~(uint32_t)(P.awp * 128 - 1);
  const uint32_t c_area = a_area + nwarps * P.awp * 128;  // awp >= kwp: aligned as well
  const uint32_t abase = a_area + warp * P.awp * 128 + lane * 4;
  const uint32_t cbase = c_area + warp * P.kwp * 128 + lane * 4;
  const uint32_t ringbase = c_area + nwarps * P.kwp * 128 + (warp * 32 + lane) * ring_stride;
  const uint32_t amask = (uint32_t)(P.awp - 1) << 7;
  const int chunks = (P.ring_mask + 1) >> 4;
  const int64_t A = T.g.aisle_len;
  const int64_t P2 = 2 * (int64_t)T.g.aisle_spacing;
  const int n8 = P.cs_pitch >> 3;  // 16-byte chunks per cursor-stream row
  for (int w = 0; w < P.aw_words; ++w) sts32(abase + w * 128, 0u);
  for (int w = 0; w < KW; ++w) sts32(cbase + w * 128, 0u);
  dep_wait();  // everything above reads only the pick table: it overlaps the segments kernel

  __shared__ unsigned long long s_task[32];
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
    int b_lo = 0, nbseg = 0;
    if (have) {
      const int nb = __ldg(nb_scratch + cand);
      b_lo = (int)((int64_t)seg * nb >> P.log2S);
      nbseg = (int)((int64_t)(seg + 1) * nb >> P.log2S) - b_lo;
    }
    const int nbmax = __reduce_max_sync(WHP_FULL, nbseg);
    uint32_t pl[kPlanes][KW];
#pragma unroll
    for (int p = 0; p < kPlanes; ++p)
#pragma unroll
      for (int w = 0; w < KW; ++w) pl[p][w] = 0;

    // ---- first batch of the segment: its start position comes from K1
    const uint32_t* __restrict__ bm = bmask + cand * P.bm_pitch;
    int p = __ldg(segstart + cand * P.ss_pitch + seg);
    int wi = p >> 5;
    uint32_t bw = __ldg(bm + wi) & (WHP_FULL << (p & 31));
    uint32_t bw_next = __ldg(bm + min(wi + 1, P.bm_pitch - 1));

    // ---- cursor stream of this lane through its private cp.async ring: chunk c (cursors of
    // positions 8c..8c+7) lives at ring offset (16 c) mod ring
    const uint4* __restrict__ cs = reinterpret_cast<const uint4*>(cstream + cand * P.cs_pitch);
    // the last chunk this lane reads: the one that holds the first position of the next segment
    // (a third of the ring traffic used to be chunks fetched past the end of the lane's run)
    int c_last;
    {
      const int p_next = __shfl_down_sync(WHP_FULL, p, 1);
      c_last = min((seg == P.S - 1 || lane == 31 ? T.n_orders : p_next) >> 3, n8 - 1);
    }
    int lo_prev;  // first chunk that was resident when the newest refill group was issued
    {
      const int c0 = p >> 3;
      for (int k = 0; k < chunks; ++k)
        if (c0 + k <= c_last) cp_async16(ringbase + (((c0 + k) << 4) & P.ring_mask), cs + c0 + k);
      cp_async_commit();
      lo_prev = c0 - chunks;
    }

    int64_t D = 0;
    uint64_t hash = 0;
    uint4 q4 = make_uint4(0u, 0u, 0u, 0u);
    for (int j = 0; j < nbmax; ++j) {
      int left = 0;  // orders of batch j
      const int p0 = p;
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
      // the newest refill group brought chunks lo_prev+chunks ..; everything older has landed
      // after wait<1>. The batch reads cursors of positions p0 .. p (one ahead).
      if (live && (p >> 3) >= lo_prev + chunks) cp_async_wait<0>(); else cp_async_wait<1>();
      // ---- the batch's picks, four records per step
      uint32_t v = 2u * (uint32_t)p0;                      // 2 x position of the next order
      const uint32_t v_end = live ? 2u * (uint32_t)p : v;
      uint32_t cur4 = lds16(ringbase + (v & P.ring_mask));  // the four being loaded
      v += live ? 2u : 0u;
      // look-ahead cursors come four at a time (one 8-byte read per four orders: a quarter of
      // the lanes take part in it, so it costs about one wavefront instead of two)
      uint32_t cw_lo, cw_hi;
      lds64(cw_lo, cw_hi, ringbase + (v & P.ring_mask & ~6u));
      auto cursor_at = [&](uint32_t vv) {  // the 16-bit cursor of position vv / 2 out of (cw_lo, cw_hi)
        return __byte_perm(cw_lo, cw_hi, (vv & 6u) * 0x11u + 0x10u) & 0xffffu;
      };
      uint32_t n_c16 = cursor_at(v);  // first four of the next order
      bool have = live;
      // (a lane without a batch keeps the four of its previous batch: its sets are discarded)
      ldg_four_if(q4, pick_f4 + 4 * (size_t)cur4, have);
      uint32_t kmax = 0, kmin = 0xffffffffu;
      uint32_t cset = 0;  // KW == 1: class set of the batch
      int m = 0;          // distinct aisles of the batch
      auto insert = [&](uint32_t rec) {
        kmax = max(kmax, rec);
        if (!DEPOT0) kmin = min(kmin, rec);
        // the distinct aisles are counted as they arrive (the close then only clears the words:
        // this kernel is bound by the L1 data pipe, and the count costs no wavefront here)
        const uint32_t aaddr = abase | ((rec >> 20) & amask);
        const uint32_t aold = lds32(aaddr), anew = aold | one_shl_wrap(rec >> 22);
        m += (anew != aold) ? 1 : 0;
        sts32(aaddr, anew);
        if (KW == 1) {
          cset |= one_shl_wrap(rec);
        } else {
          const uint32_t caddr = cbase | (rec & 0x380u);
          sts32(caddr, lds32(caddr) | one_shl_wrap(rec));
        }
      };
      while (__any_sync(WHP_FULL, have)) {
        const uint32_t r0 = q4.x, r1 = q4.y, r2 = q4.z, r3 = q4.w;
        // where the next four is: the next one of this order, the first one of the next order,
        // or nowhere (then the lane stays on this four)
        const bool last4 = (r3 & WHP_FAST_LAST4) != 0u;
        const bool next_order = last4 && (v != v_end);
        have = have && (!last4 || next_order);
        cur4 = next_order ? n_c16 : cur4 + 1u;
        v += next_order ? 2u : 0u;
        lds64_if(cw_lo, cw_hi, ringbase + (v & P.ring_mask), next_order && (v & 6u) == 0u);
        n_c16 = cursor_at(v);
        ldg_four_if(q4, pick_f4 + 4 * (size_t)cur4, have);
        insert(r0); insert(r1); insert(r2); insert(r3);
      }
      {  // refill the slots of the chunks this batch finished; waited for two batches later
        const int nf = live ? (p >> 3) - (p0 >> 3) : 0;
        const int nfmax = __reduce_max_sync(WHP_FULL, nf);
        for (int i = 0; i < nfmax; ++i) {
          const int c = (p0 >> 3) + i;
          if (i < nf && c + chunks <= c_last) cp_async16(ringbase + ((c << 4) & P.ring_mask), cs + c + chunks);
        }
        cp_async_commit();
        if (live) lo_prev = p0 >> 3;
      }
      // ---- close the batch: m = distinct aisles, D4; the sets are emptied for the next batch
#pragma unroll 4
      for (int w = 0; w < P.aw_words; ++w) sts32(abase + w * 128, 0u);
      if (live) {
        const uint32_t a_max = WHP_FAST_AISLE(kmax);
        const uint32_t slot1 = WHP_FAST_SLOT1(kmax);
        if (DEPOT0 && P.fits32) {
          const uint32_t d2 = 2u * slot1 * (uint32_t)T.g.slot_pitch;
          D += (uint32_t)P2 * a_max + (uint32_t)m * (uint32_t)A + ((m & 1) ? d2 - (uint32_t)A : 0u);
        } else {
          const int64_t d_last = (int64_t)slot1 * T.g.slot_pitch;
          int64_t H;
          if (DEPOT0) {
            H = P2 * (int64_t)a_max;
          } else {
            const int64_t a_min = WHP_FAST_AISLE(kmin), a0 = T.g.depot_aisle;
            H = (int64_t)T.g.aisle_spacing *
                (llabs(a0 - a_min) + ((int64_t)a_max - a_min) + llabs((int64_t)a_max - a0));
          }
          D += H + ((m & 1) ? (int64_t)(m - 1) * A + 2 * d_last : (int64_t)m * A);
        }
      }
      // the batch's class set goes into the vertical counters (D5)
#pragma unroll
      for (int w = 0; w < KW; ++w) {
        // lanes without a batch j ran the steps on a dummy pick: their set is discarded
        uint32_t carry;
        if (KW == 1) {
          carry = cset;
        } else {
          carry = lds32(cbase + w * 128);
          sts32(cbase + w * 128, 0u);
        }
        if (!live) carry = 0u;
#pragma unroll
        for (int pp = 0; pp < kPlanes; ++pp) {
          const uint32_t t2 = pl[pp][w] & carry;
          pl[pp][w] ^= carry;
          carry = t2;
        }
      }
    }
    cp_async_wait<0>();  // nothing of this task may still land in the ring
    // ---- combine the S segment lanes of each candidate (D, hash); write the counters
#pragma unroll
    for (int o = 1; o < 32; o <<= 1)
      if (o < P.S) {
        D += __shfl_xor_sync(WHP_FULL, D, o);
        hash += __shfl_xor_sync(WHP_FULL, hash, o);
      }
    const bool fused = P.S == 32;  // the warp is one plan: it finishes D6 itself (no K3)
    if (have && seg == 0) {
      if (!fused) dist_scratch[cand] = D;
      if (hash_out) hash_out[cand] = hash;
    }
    double phi = 0.0;
    // bit-sliced addition of the S lanes' vertical counters (one more plane per level)
    {
      uint32_t* __restrict__ po = planes_out + cand * (kPlaneRow * KW);
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
        if (fused) {
          // every lane holds the plan's counters: lane l decodes r_k of class 32w + l and adds
          // its term — ascending w, lane = k mod 32: the canonical accumulation of D6
          uint32_t r = 0;
#pragma unroll
          for (int pp = 0; pp < kPlanes + 5; ++pp) r |= ((a[pp] >> lane) & 1u) << pp;
          const int k = 32 * w + lane;
          if (k < T.K) {
            if (o_resp && have) o_resp[cand * T.K + k] = (int32_t)r;
            const double c = __dsub_rn(__ldg(T.tvw + k), (double)r);
            const double u = __dmul_rn(__ldg(T.tvw + 2 * T.K + k), c);
            phi = __dadd_rn(phi, __dadd_rn(__dmul_rn(__ldg(T.tvw + T.K + k), c), __dmul_rn(u, u)));
          }
        } else if (have && seg == 0) {
#pragma unroll
          for (int pp = 0; pp < kPlanes + 5; ++pp)
            if (pp < kPlanes + P.log2S) po[pp * KW + w] = a[pp];
        }
      }
    }
    if (fused) {
#pragma unroll
      for (int off = 16; off >= 1; off >>= 1) phi = __dadd_rn(phi, __shfl_xor_sync(WHP_FULL, phi, off));
      if (have && lane == 0) {
        if (o_dist) o_dist[cand] = D;
        if (o_pen) o_pen[cand] = phi;
        if (o_obj) o_obj[cand] = __dadd_rn((double)D, phi);
      }
    }
    __syncwarp();
  }
}

// ------------------------------------------------------------------------------------------ KL
// NEXT-2 tuned: leg sums (reading N2) on the K1 outputs. Same decomposition as K2 — one lane per
// (plan, segment), one pick per branch-free step — but a step only adds the leg from the previous
// pick (D0's walking metric); there are no sets. A cart starts and ends at the depot; a lane
// that has finished its cart stays on its last pick (a zero leg).
template <bool SMEM_TABLES, bool FOURS>
__global__ void __launch_bounds__(1024, 1)
whp_legs_kernel(const whp_tables T, const sets_params P, const uint32_t* __restrict__ pick_fast,
                const uint16_t* __restrict__ cstream, const uint32_t* __restrict__ bmask,
                const int32_t* __restrict__ nb_scratch, const int32_t* __restrict__ segstart,
                int64_t n_cand, int64_t* __restrict__ len_out,
                unsigned long long* __restrict__ task_counter) {
  extern __shared__ __align__(16) uint32_t smem[];
  uint32_t* priv = smem;
  uint32_t pick_base = 0;
  if (SMEM_TABLES) {
    for (int i = threadIdx.x; i < P.n_items_pad; i += blockDim.x) smem[i] = __ldg(pick_fast + i);
    pick_base = smem_u32(smem);
    priv = smem + ((P.n_items_pad + 31) & ~31);
    __syncthreads();
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ring_stride = P.ring_mask + 1 + 16;
  const uint32_t ringbase = smem_u32(priv) + (warp * 32 + lane) * ring_stride;
  uint32_t pb;
  asm volatile("mov.u32 %0, %1;" : "=r"(pb) : "r"(pick_base));
  const int chunks = (P.ring_mask + 1) >> 4;
  const int Cmax = T.C;
  const int n8 = P.cs_pitch >> 3;
  const int32_t a0 = T.g.depot_aisle;
  const int64_t A2 = 2 * T.g.aisle_len, Psp = T.g.aisle_spacing, pitch = T.g.slot_pitch;

  __shared__ unsigned long long s_task[32];
  for (;;) {
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
    int nbseg = 0;
    if (have) {
      const int nb = __ldg(nb_scratch + cand);
      const int b_lo = (int)((int64_t)seg * nb >> P.log2S);
      nbseg = (int)((int64_t)(seg + 1) * nb >> P.log2S) - b_lo;
    }
    const int nbmax = __reduce_max_sync(WHP_FULL, nbseg);
    const uint32_t* __restrict__ bm = bmask + cand * P.bm_pitch;
    int p = __ldg(segstart + cand * P.ss_pitch + seg);
    int wi = p >> 5;
    uint32_t bw = __ldg(bm + wi) & (WHP_FULL << (p & 31));
    uint32_t bw_next = __ldg(bm + min(wi + 1, P.bm_pitch - 1));
    const uint4* __restrict__ cs = reinterpret_cast<const uint4*>(cstream + cand * P.cs_pitch);
    int c_last;  // the last chunk this lane reads (as in K2)
    {
      const int p_next = __shfl_down_sync(WHP_FULL, p, 1);
      c_last = min((seg == P.S - 1 || lane == 31 ? T.n_orders : p_next) >> 3, n8 - 1);
    }
    int lo_prev;
    {
      const int c0 = p >> 3;
      for (int k = 0; k < chunks; ++k)
        if (c0 + k <= c_last) cp_async16(ringbase + (((c0 + k) << 4) & P.ring_mask), cs + c0 + k);
      cp_async_commit();
      lo_prev = c0 - chunks;
    }
    int64_t L = 0;
    uint4 q4 = make_uint4(0u, 0u, 0u, 0u);
    for (int j = 0; j < nbmax; ++j) {
      int left = 0;
      const int p0 = p;
      if (j < nbseg) {
        bw &= bw - 1;
        while (bw == 0) {
          ++wi;
          bw = bw_next;
          bw_next = __ldg(bm + min(wi + 1, P.bm_pitch - 1));
        }
        const int pe = 32 * wi + __ffs(bw) - 1;
        left = pe - p;
        p = pe;
      }
      const bool live = left > 0;
      if (live && (p >> 3) >= lo_prev + chunks) cp_async_wait<0>(); else cp_async_wait<1>();
      // the cart sets out from the depot
      int32_t pa = a0;
      int64_t py = 0, Lb = 0;
      uint32_t Lb32 = 0;
      int32_t py32 = 0;
      auto walk = [&](uint32_t rec) {  // the leg from the previous point to this pick
        const int32_t a = (int32_t)WHP_FAST_AISLE(rec);
        if (P.fits32) {
          const int32_t y = (int32_t)WHP_FAST_SLOT1(rec) * (int32_t)pitch;
          const int32_t da = abs(a - pa);
          const int32_t front = y + py32, back = (int32_t)A2 - front;
          const int32_t cross = da * (int32_t)Psp + min(front, back);
          Lb32 += (uint32_t)(da == 0 ? abs(y - py32) : cross);
          py32 = y;
        } else {
          const int64_t y = (int64_t)WHP_FAST_SLOT1(rec) * pitch;
          const int64_t da = llabs((int64_t)a - pa);
          const int64_t front = y + py, back = A2 - front;
          Lb += da == 0 ? llabs(y - py) : da * Psp + (front < back ? front : back);
          py = y;
        }
        pa = a;
      };
      if (FOURS) {
        // the four-aligned table (as in whp_sets4_kernel): a step is one 16-byte load = four picks;
        // padding copies and a lane whose cart is exhausted walk to the point they stand on
        uint32_t v = 2u * (uint32_t)p0;
        const uint32_t v_end = live ? 2u * (uint32_t)p : v;
        uint32_t cur4 = lds16(ringbase + (v & P.ring_mask));
        v += live ? 2u : 0u;
        uint32_t n_c16 = lds16(ringbase + (v & P.ring_mask));
        bool fresh = live;  // q4 holds (or is about to receive) a four that has not been walked
        uint32_t stay = 0;  // the last pick walked
        ldg_four_if(q4, pick_fast + 4 * (size_t)cur4, fresh);
        while (__any_sync(WHP_FULL, fresh)) {
          const uint32_t r0 = fresh ? q4.x : stay, r1 = fresh ? q4.y : stay;
          const uint32_t r2 = fresh ? q4.z : stay, r3 = fresh ? q4.w : stay;
          stay = r3;
          const bool last4 = (r3 & WHP_FAST_LAST4) != 0u;
          const bool next_order = last4 && (v != v_end);
          fresh = fresh && (!last4 || next_order);
          cur4 = next_order ? n_c16 : cur4 + 1u;
          v += next_order ? 2u : 0u;
          lds16_if(n_c16, ringbase + (v & P.ring_mask), next_order);
          ldg_four_if(q4, pick_fast + 4 * (size_t)cur4, fresh);
          walk(r0); walk(r1); walk(r2); walk(r3);
        }
      } else {
        uint32_t v = live ? 2u * (uint32_t)p0 : 0u;
        const uint32_t v_end = live ? 2u * (uint32_t)p : 0u;
        uint32_t cur;
        if (live) {
          const uint32_t c16 = lds16(ringbase + (v & P.ring_mask));
          cur = SMEM_TABLES ? pb + 8 * c16 : 2 * c16;
          v += 2;
        } else {
          cur = SMEM_TABLES ? pb : 0u;
        }
        uint32_t n_c16 = lds16(ringbase + (v & P.ring_mask));
        uint32_t rec = SMEM_TABLES ? lds32(cur) : __ldg(pick_fast + cur);
  #pragma unroll 2
        for (int t = 0; t < Cmax; ++t) {
          const uint32_t first_of_next = SMEM_TABLES ? pb + 8 * n_c16 : 2 * n_c16;
          const bool last = (int32_t)(rec << 26) < 0;
          const bool more = last && (v != v_end);
          uint32_t nxt = last ? cur : cur + (SMEM_TABLES ? 4u : 1u);
          nxt = more ? first_of_next : nxt;
          v = more ? v + 2 : v;
          lds16_if(n_c16, ringbase + (v & P.ring_mask), more);
          cur = nxt;
          const uint32_t rec_next = SMEM_TABLES ? lds32(cur) : __ldg(pick_fast + cur);
          walk(rec);
          rec = rec_next;
        }
      }
      {
        const int nf = live ? (p >> 3) - (p0 >> 3) : 0;
        const int nfmax = __reduce_max_sync(WHP_FULL, nf);
        for (int i = 0; i < nfmax; ++i) {
          const int c = (p0 >> 3) + i;
          if (i < nf && c + chunks <= c_last) cp_async16(ringbase + ((c << 4) & P.ring_mask), cs + c + chunks);
        }
        cp_async_commit();
        if (live) lo_prev = p0 >> 3;
      }
      if (live) {  // the way home, and the cart's total (a lane without a cart walked a dummy)
        if (P.fits32) {
          const int32_t da = abs(pa - a0);
          L += (int64_t)Lb32 + (da == 0 ? py32 : da * (int32_t)Psp + py32);
        } else {
          const int64_t da = llabs((int64_t)pa - a0);
          L += Lb + (da == 0 ? py : da * Psp + py);
        }
      }
    }
    cp_async_wait<0>();
#pragma unroll
    for (int o = 1; o < 32; o <<= 1)
      if (o < P.S) L += __shfl_xor_sync(WHP_FULL, L, o);
    if (have && seg == 0) len_out[cand] = L;
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
  // the candidate's counter words are read by broadcast loads (every lane needs its own bit of
  // every word): plane pp of class word w holds bit pp of r_k for the 32 classes of that word
  const uint32_t* __restrict__ pc = planes + cand * (kPlaneRow * KW);
  double s = 0.0;
  const int kw_used = (T.K + 31) >> 5;
  for (int w = 0; w < kw_used; ++w) {
    int r = 0;
    if (planes_used == 0) {  // K2 already decoded the counters (S = 32)
      r = (int)__ldg(reinterpret_cast<const uint16_t*>(pc) + 32 * w + lane);
    } else {
#pragma unroll 4
      for (int pp = 0; pp < planes_used; ++pp)
        r |= (int)((__ldg(pc + pp * KW + w) >> lane) & 1u) << pp;
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

// upper bound on the number of batches of any plan (derived in whp_load_orders)
static int64_t nb_upper_bound(const whp_ctx* c) { return c->nb_ub; }

static int bounds_stages(int warps) { return warps == 5 ? kStagesWide : kStages; }
static size_t bounds_smem_bytes(const whp_ctx* c, int warps = 1) {
  const int st = bounds_stages(warps);
  return 1024 + (size_t)warps * (st + 2) * kTileBytes +
         4 * (((size_t)c->n_orders + 3) & ~(size_t)3) + 8 * ((size_t)warps * st + 1);
}
// K1 wants four resident warps per SM (one per scheduler): blocks of one warp when four of
// them fit, else two or four warps that share one copy of the order table
static int bounds_warps(const whp_ctx* c, int64_t n_cand) {
  const size_t cap = (size_t)c->smem_optin;
  if (c->dbg_k1_warps == 1 || c->dbg_k1_warps == 2 || c->dbg_k1_warps == 4 || c->dbg_k1_warps == 5)  // WHP_DEBUG_K1_WARPS
    if (bounds_smem_bytes(c, c->dbg_k1_warps) + 1024 <= cap) return c->dbg_k1_warps;
  if (4 * (bounds_smem_bytes(c, 1) + 1024) <= cap) return 1;
  if (2 * (bounds_smem_bytes(c, 2) + 1024) <= cap) return 2;
  // one block per SM: when the launch takes several waves of four-warp blocks, five warps with
  // five tiles in flight each make the waves fewer (a warp's time is set by its plan's serial
  // recurrence, not by the tiles in flight: stress scale 4 -> 3 waves)
  if (bounds_smem_bytes(c, 5) + 1024 <= cap && n_cand > 128ll * c->num_sms) return 5;
  if (bounds_smem_bytes(c, 4) + 1024 <= cap) return 4;
  if (bounds_smem_bytes(c, 2) + 1024 <= cap) return 2;
  return 1;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
static PFN_cuTensorMapEncodeTiled tensor_map_encoder() {
  static PFN_cuTensorMapEncodeTiled fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (PFN_cuTensorMapEncodeTiled)p;
  }
  return fn;
}

bool whp_fast_eligible(const whp_ctx* c) {
  if (!c->fast_tables_ok) return false;                       // cursors must fit 16 bits
  if (c->n_orders >= 65536) return false;
  if ((nb_upper_bound(c) + 31) / 32 > 255) return false;      // 8 counter planes, S <= 32
  if ((c->C + 14) / 8 + 1 > 16) return false;                // per-lane cursor ring of 16 chunks (C <= 106)
  if (bounds_smem_bytes(c) > (size_t)c->smem_optin - 1024) return false;  // K1: order table in smem
  return true;
}

static int32_t fast_bm_pitch(const whp_ctx* c) { return (int32_t)((((c->n_orders + 31) >> 5) + 2 + 3) & ~3); }
static int32_t fast_cs_pitch(const whp_ctx* c) { return (int32_t)((c->n_orders + 7) & ~7); }
constexpr int32_t kSsPitch = 32;

// scratch of the tuned paths (grow-only; reallocated when the shape changes)
static cudaError_t ensure_fast_scratch(whp_ctx* c, int64_t n_cand, int64_t plane_words, cudaStream_t st) {
  const int32_t bm_pitch = fast_bm_pitch(c), cs_pitch = fast_cs_pitch(c), ss_pitch = kSsPitch;
  if (c->fast_cap < n_cand || c->fast_pitch != bm_pitch || c->fast_plane_words < plane_words) {
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    cudaFree(c->d_bmask); cudaFree(c->d_cstream); cudaFree(c->d_nb); cudaFree(c->d_dist_scratch);
    cudaFree(c->d_planes); cudaFree(c->d_segstart);
    c->d_bmask = nullptr; c->d_cstream = nullptr; c->d_nb = nullptr; c->d_dist_scratch = nullptr;
    c->d_planes = nullptr; c->d_segstart = nullptr;
    const int64_t cap = n_cand > c->fast_cap ? n_cand : c->fast_cap;
    const int64_t pw = plane_words > c->fast_plane_words ? plane_words : c->fast_plane_words;
    c->fast_cap = 0;
    if ((e = cudaMalloc(&c->d_bmask, 4 * (size_t)cap * bm_pitch)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_cstream, 2 * (size_t)cap * cs_pitch + 64)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_nb, 4 * (size_t)cap)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_dist_scratch, 8 * (size_t)cap)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_planes, 4 * (size_t)cap * pw)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&c->d_segstart, 4 * (size_t)cap * ss_pitch)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(c->d_bmask, 0, 4 * (size_t)cap * bm_pitch, st)) != cudaSuccess) return e;
    c->fast_cap = cap; c->fast_pitch = bm_pitch; c->fast_plane_words = pw;
  }
  return cudaSuccess;
}

// K1 (batch boundaries, cursor stream) and the segment starts of every plan
static cudaError_t launch_bounds_and_segments(whp_ctx* c, const void* d_perms, int64_t n_cand, int S,
                                              int log2S, int32_t* n_batches_out, cudaStream_t st,
                                              bool perm16 = false, const uint32_t* order_table = nullptr) {
  if (!order_table) order_table = c->d_order_fast;  // else: cursors of the four-aligned layout
  const int32_t bm_pitch = fast_bm_pitch(c), cs_pitch = fast_cs_pitch(c), ss_pitch = kSsPitch;
  {
    // (Folding this reset into the segments kernel saves 1 us of the evaluation alone and costs
    // 13 us of bench.py's two-stream step: K1 then reaches the SMs before the other stream's
    // one-block base kernel, whose 92 KB of shared memory no longer fit beside K1's blocks.)
    cudaError_t e = cudaMemsetAsync(c->d_task, 0, 2 * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    const int kw1 = bounds_warps(c, n_cand);
    const size_t smem = bounds_smem_bytes(c, kw1);
    // tensor map over this call's permutation matrix: [n_cand][n_orders] int32, box 32 x 32
    PFN_cuTensorMapEncodeTiled encode = tensor_map_encoder();
    if (!encode) return cudaErrorNotSupported;
    // TMA needs a 16-byte aligned matrix with a row pitch that is a multiple of 16 bytes:
    // otherwise the plans are first copied into a padded scratch matrix
    const size_t elem = perm16 ? 2 : 4;  // bytes of an order id
    size_t pitch_bytes = elem * (size_t)c->n_orders;
    if ((pitch_bytes & 15u) != 0 || ((uintptr_t)d_perms & 15u) != 0) {
      pitch_bytes = (pitch_bytes + 15) & ~(size_t)15;
      if (c->perm_pad_bytes < pitch_bytes * (size_t)n_cand) {
        if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return e;
        cudaFree(c->d_perm_pad);
        c->d_perm_pad = nullptr;
        c->perm_pad_bytes = 0;
        if ((e = cudaMalloc(&c->d_perm_pad, pitch_bytes * (size_t)n_cand)) != cudaSuccess) return e;
        c->perm_pad_bytes = pitch_bytes * (size_t)n_cand;
      }
      if ((e = cudaMemcpy2DAsync(c->d_perm_pad, pitch_bytes, d_perms, elem * (size_t)c->n_orders,
                                 elem * (size_t)c->n_orders, (size_t)n_cand, cudaMemcpyDeviceToDevice,
                                 st)) != cudaSuccess)
        return e;
      d_perms = c->d_perm_pad;
    }
    CUtensorMap tmap;
    const cuuint64_t gdim[2] = {(cuuint64_t)c->n_orders, (cuuint64_t)n_cand};
    const cuuint64_t gstride[1] = {(cuuint64_t)pitch_bytes};
    const cuuint32_t box[2] = {perm16 ? 64u : 32u, 32};  // 128 bytes x 32 plans
    const cuuint32_t estr[2] = {1, 1};
    if (encode(&tmap, perm16 ? CU_TENSOR_MAP_DATA_TYPE_UINT16 : CU_TENSOR_MAP_DATA_TYPE_INT32, 2,
               (void*)d_perms, gdim, gstride, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
               CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
    // tensor map over the cursor stream: [n_cand][cs_pitch] u16, box 32 rows x 64 cursors
    CUtensorMap tmap_cs;
    const cuuint64_t cdim[2] = {(cuuint64_t)cs_pitch, (cuuint64_t)n_cand};
    const cuuint64_t cstride[1] = {2ull * (cuuint64_t)cs_pitch};
    const cuuint32_t cbox[2] = {64, 32};
    if (encode(&tmap_cs, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, (void*)c->d_cstream, cdim, cstride, cbox,
               estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
               CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
    const unsigned blocks = (unsigned)((n_cand + 32 * kw1 - 1) / (32 * kw1));
#define WHP_LAUNCH_BOUNDS_T(KW1, U16V)                                                          \
  do {                                                                                          \
    constexpr int kSt_ = KW1 == 5 ? kStagesWide : kStages;                                      \
    cudaFuncSetAttribute(whp_bounds_kernel<KW1, U16V, kSt_>,                                    \
                         cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin - 1024);    \
    whp_bounds_kernel<KW1, U16V, kSt_><<<blocks, 32 * KW1, smem, st>>>(                         \
        tmap, tmap_cs, order_table, c->n_orders, c->C, n_cand, c->d_bmask, bm_pitch,            \
        c->d_cstream, cs_pitch);                                                                \
  } while (0)
#define WHP_LAUNCH_BOUNDS(KW1)                                                                  \
  do {                                                                                          \
    if (perm16) WHP_LAUNCH_BOUNDS_T(KW1, true); else WHP_LAUNCH_BOUNDS_T(KW1, false);           \
  } while (0)
    if (kw1 == 1) WHP_LAUNCH_BOUNDS(1);
    else if (kw1 == 2) WHP_LAUNCH_BOUNDS(2);
    else if (kw1 == 5) WHP_LAUNCH_BOUNDS(5);
    else WHP_LAUNCH_BOUNDS(4);
#undef WHP_LAUNCH_BOUNDS_T
#undef WHP_LAUNCH_BOUNDS
    c->launches += 1;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    whp_segments_kernel<<<(unsigned)((n_cand * 32 + 255) / 256), 256, 0, st>>>(
        c->d_bmask, bm_pitch, c->n_orders, n_cand, S, log2S, c->d_nb, n_batches_out,
        c->d_segstart, ss_pitch);
    c->launches += 1;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t whp_launch_eval_fast(whp_ctx* c, const void* d_perms, int64_t n_cand,
                                 const whp_eval_out& out, cudaStream_t st, bool perm16) {
  const whp_tables T = whp_make_tables(c);
  const int64_t nb_ub = nb_upper_bound(c);
  const int32_t bm_pitch = fast_bm_pitch(c), cs_pitch = fast_cs_pitch(c), ss_pitch = kSsPitch;
  const int KW = c->K <= 32 ? 1 : c->K <= 64 ? 2 : c->K <= 128 ? 4 : c->K <= 224 ? 7 : 8;
  const int aw_words = (c->g.n_aisles + 31) / 32;
  // cursor ring: a batch of C orders touches at most (C+14)/8 chunks of 8 cursors, and the
  // cursor one past its end is read too
  const int ring_bytes = ((c->C + 14) / 8 + 1 <= 8) ? 128 : 256;
  // K2 shape
  const size_t table_bytes = 4 * (((size_t)c->n_items_pad + 31) & ~(size_t)31);
  int awp = 1, kwp = 1;
  while (awp < aw_words) awp <<= 1;
  while (kwp < KW) kwp <<= 1;
  if (awp < kwp) awp = kwp;
  const size_t priv_per_warp = (size_t)(kwp + awp) * 128 + 32 * (size_t)(ring_bytes + 16);
  const size_t smem_max = (size_t)c->smem_optin - 1024 - (size_t)awp * 128;  // alignment slack
  const bool smem_tables = table_bytes + 4 * priv_per_warp <= smem_max;
  // tables beyond shared memory: the four-aligned layout (K2')
  const bool fours = !smem_tables && c->d_pick_f4 != nullptr && !c->dbg_no_fours;
  const size_t avail = smem_max - (smem_tables ? table_bytes : 0);
  // segments: few enough batches per segment for the counter planes, and >= 4 tasks per warp
  int warps_cap = 24;
  int S = 1;
  while (S < 32 && ((nb_ub + S - 1) / S > 255 || n_cand * S < 4ll * c->num_sms * warps_cap * 32)) S <<= 1;
  // every plan has at least n_items / C batches: with eight or more per lane a warp is one plan
  // (S = 32) whatever the plan count, so K2 finishes D6 itself — no K3 launch and no counter
  // round trip (stress scale: 9.79 -> 9.58 ms against S = 8)
  if ((int64_t)c->n_items / c->C >= 256) S = 32;
  if (c->dbg_segments >= 1) {  // whp_debug_set(WHP_DEBUG_SEGMENTS): ignored when not legal
    const int v = c->dbg_segments;
    if (v <= 32 && (v & (v - 1)) == 0 && (nb_ub + v - 1) / v <= 255) S = v;
  }
  int log2S = 0;
  while ((1 << log2S) < S) ++log2S;
  int seg_planes = 1;  // planes of one segment's counters; one more per combine level
  while ((1ll << seg_planes) <= (nb_ub + S - 1) / S) ++seg_planes;
  const int kernel_planes = seg_planes <= 4 ? 4 : seg_planes <= 6 ? 6 : 8;  // the instantiation
  if (KW * kernel_planes > (fours ? 16 : 42)) warps_cap = 16;  // __launch_bounds__ of the register-heavy instantiations
  int warps = (int)(avail / priv_per_warp);
  if (warps > warps_cap) warps = warps_cap;
  if (c->dbg_warps >= 1 && c->dbg_warps <= warps) warps = c->dbg_warps;  // WHP_DEBUG_WARPS
  if (warps < 1) return cudaErrorInvalidConfiguration;
  const int planes_used = kernel_planes + log2S;
  // every per-batch length below 2^31: the close can work in 32 bits
  const int64_t worst = 2ll * c->g.aisle_spacing * c->g.n_aisles +
                        ((int64_t)c->g.n_aisles + 2) * c->g.aisle_len;
  const int fits32 = worst < (1ll << 31) ? 1 : 0;
  cudaError_t e0 = ensure_fast_scratch(c, n_cand, (int64_t)kPlaneRow * KW, st);
  if (e0 != cudaSuccess) return e0;
  if ((e0 = launch_bounds_and_segments(c, d_perms, n_cand, S, log2S, out.n_batches, st, perm16,
                                       fours ? c->d_order_fast4 : nullptr)) != cudaSuccess)
    return e0;
  // K2
  {
    sets_params P;
    P.S = S; P.log2S = log2S;
    P.aw_words = aw_words; P.awp = awp; P.kwp = kwp; P.ring_mask = ring_bytes - 1;
    P.bm_pitch = bm_pitch; P.cs_pitch = cs_pitch; P.ss_pitch = ss_pitch;
    P.n_items_pad = c->n_items_pad; P.fits32 = fits32;
    P.n_tasks = (n_cand * S + 31) / 32;
    int64_t blocks = (P.n_tasks + warps - 1) / warps;
    if (blocks > c->num_sms) blocks = c->num_sms;
    const size_t smem = (smem_tables ? table_bytes : 0) + priv_per_warp * warps + (size_t)awp * 128;
    const bool depot0 = c->g.depot_aisle == 0;
#define WHP_LAUNCH_SETS_PL(ST, D0, KWV, PLV)                                                     \
  do {                                                                                           \
    cudaFuncSetAttribute(whp_sets_kernel<ST, D0, KWV, PLV>,                                      \
                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(c->smem_optin - 1024)); \
    cudaLaunchConfig_t cfg{};                                                                    \
    cfg.gridDim = dim3((unsigned)blocks);                                                        \
    cfg.blockDim = dim3(warps * 32);                                                             \
    cfg.dynamicSmemBytes = smem;                                                                 \
    cfg.stream = st;                                                                             \
    cudaLaunchAttribute attr[1];                                                                 \
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;                             \
    attr[0].val.programmaticStreamSerializationAllowed = 1;                                      \
    cfg.attrs = attr;                                                                            \
    cfg.numAttrs = 1;                                                                            \
    cudaLaunchKernelEx(&cfg, whp_sets_kernel<ST, D0, KWV, PLV>, T, P,                            \
                       (const uint32_t*)c->d_pick_fast, (const uint16_t*)c->d_cstream,           \
                       (const uint32_t*)c->d_bmask, (const int32_t*)c->d_nb,                     \
                       (const int32_t*)c->d_segstart, n_cand, c->d_dist_scratch, c->d_planes,    \
                       out.batch_hash, c->d_task, out.dist, out.penalty, out.obj, out.resp);     \
  } while (0)
#define WHP_LAUNCH_SETS(ST, D0, KWV)                                                             \
  do {                                                                                           \
    if (kernel_planes == 4) WHP_LAUNCH_SETS_PL(ST, D0, KWV, 4);                                  \
    else if (kernel_planes == 6) WHP_LAUNCH_SETS_PL(ST, D0, KWV, 6);                             \
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
#define WHP_LAUNCH_SETS4_PL(D0, KWV, PLV)                                                        \
  do {                                                                                           \
    cudaFuncSetAttribute(whp_sets4_kernel<D0, KWV, PLV>,                                         \
                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(c->smem_optin - 1024)); \
    cudaLaunchConfig_t cfg{};                                                                    \
    cfg.gridDim = dim3((unsigned)blocks);                                                        \
    cfg.blockDim = dim3(warps * 32);                                                             \
    cfg.dynamicSmemBytes = smem;                                                                 \
    cfg.stream = st;                                                                             \
    cudaLaunchAttribute attr[1];                                                                 \
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;                             \
    attr[0].val.programmaticStreamSerializationAllowed = 1;                                      \
    cfg.attrs = attr;                                                                            \
    cfg.numAttrs = 1;                                                                            \
    cudaLaunchKernelEx(&cfg, whp_sets4_kernel<D0, KWV, PLV>, T, P,                               \
                       (const uint32_t*)c->d_pick_f4,                                            \
                       (const uint16_t*)c->d_cstream, (const uint32_t*)c->d_bmask,               \
                       (const int32_t*)c->d_nb, (const int32_t*)c->d_segstart, n_cand,           \
                       c->d_dist_scratch, c->d_planes, out.batch_hash, c->d_task, out.dist,      \
                       out.penalty, out.obj, out.resp);                                          \
  } while (0)
#define WHP_LAUNCH_SETS4(D0, KWV)                                                                \
  do {                                                                                           \
    if (kernel_planes == 4) WHP_LAUNCH_SETS4_PL(D0, KWV, 4);                                     \
    else if (kernel_planes == 6) WHP_LAUNCH_SETS4_PL(D0, KWV, 6);                                \
    else WHP_LAUNCH_SETS4_PL(D0, KWV, 8);                                                        \
  } while (0)
#define WHP_LAUNCH_SETS4_KW(D0)                                                                  \
  do {                                                                                           \
    if (KW == 1) WHP_LAUNCH_SETS4(D0, 1);                                                        \
    else if (KW == 2) WHP_LAUNCH_SETS4(D0, 2);                                                   \
    else if (KW == 4) WHP_LAUNCH_SETS4(D0, 4);                                                   \
    else if (KW == 7) WHP_LAUNCH_SETS4(D0, 7);                                                   \
    else WHP_LAUNCH_SETS4(D0, 8);                                                                \
  } while (0)
    if (fours && depot0) WHP_LAUNCH_SETS4_KW(true);
    else if (fours) WHP_LAUNCH_SETS4_KW(false);
    else if (smem_tables && depot0) WHP_LAUNCH_SETS_KW(true, true);
    else if (smem_tables) WHP_LAUNCH_SETS_KW(true, false);
    else if (depot0) WHP_LAUNCH_SETS_KW(false, true);
    else WHP_LAUNCH_SETS_KW(false, false);
#undef WHP_LAUNCH_SETS_KW
#undef WHP_LAUNCH_SETS
#undef WHP_LAUNCH_SETS_PL
#undef WHP_LAUNCH_SETS4_KW
#undef WHP_LAUNCH_SETS4
#undef WHP_LAUNCH_SETS4_PL
    c->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  if (out.batch_of_pos) {
    whp_bop_kernel<<<(unsigned)((n_cand * 32 + 255) / 256), 256, 0, st>>>(
        c->d_bmask, bm_pitch, c->n_orders, n_cand, out.batch_of_pos);
    c->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  // K3
  if (S != 32 && (out.dist || out.penalty || out.obj || out.resp)) {  // S = 32: K2 finished D6 itself
    const unsigned blocks = (unsigned)((n_cand * 32 + 255) / 256);
    whp_finish_kernel<<<blocks, 256, 0, st>>>(T, n_cand, c->d_dist_scratch, c->d_planes, KW,
                                              S == 32 ? 0 : planes_used, out.dist, out.penalty, out.obj,
                                              out.resp);
    c->launches += 1;
    return cudaGetLastError();
  }
  return cudaSuccess;
}

// NEXT-2 on the tuned infrastructure: K1 + segments, then the leg kernel
cudaError_t whp_launch_legsum_fast(whp_ctx* c, const int32_t* d_perms, int64_t n_cand, int64_t* d_len,
                                   cudaStream_t st) {
  const whp_tables T = whp_make_tables(c);
  const int64_t nb_ub = nb_upper_bound(c);
  const int ring_bytes = ((c->C + 14) / 8 + 1 <= 8) ? 128 : 256;
  const size_t table_bytes = 4 * (((size_t)c->n_items_pad + 31) & ~(size_t)31);
  const size_t priv_per_warp = 32 * (size_t)(ring_bytes + 16);
  const size_t smem_max = (size_t)c->smem_optin - 1024;
  const bool smem_tables = table_bytes + 4 * priv_per_warp <= smem_max;
  int warps = (int)((smem_max - (smem_tables ? table_bytes : 0)) / priv_per_warp);
  if (warps > 32) warps = 32;
  if (warps < 1) return cudaErrorInvalidConfiguration;
  int S = 1;
  while (S < 32 && n_cand * S < 4ll * c->num_sms * warps * 32) S <<= 1;
  int log2S = 0;
  while ((1 << log2S) < S) ++log2S;
  (void)nb_ub;
  // a cart's legs in 32 bits: at most C + 1 legs, each below spacing * aisles + 2 * aisle length
  const int64_t worst = ((int64_t)c->C + 2) * ((int64_t)c->g.aisle_spacing * c->g.n_aisles + 2 * c->g.aisle_len);
  cudaError_t e = ensure_fast_scratch(c, n_cand, 0, st);
  if (e != cudaSuccess) return e;
  const bool fours = !smem_tables && c->d_pick_f4 != nullptr && !c->dbg_no_fours;  // as in K2'
  if ((e = launch_bounds_and_segments(c, d_perms, n_cand, S, log2S, nullptr, st, false,
                                      fours ? c->d_order_fast4 : nullptr)) != cudaSuccess) return e;
  sets_params P{};
  P.S = S; P.log2S = log2S; P.ring_mask = ring_bytes - 1;
  P.bm_pitch = fast_bm_pitch(c); P.cs_pitch = fast_cs_pitch(c); P.ss_pitch = kSsPitch;
  P.n_items_pad = c->n_items_pad; P.fits32 = worst < (1ll << 31) ? 1 : 0;
  P.n_tasks = (n_cand * S + 31) / 32;
  int64_t blocks = (P.n_tasks + warps - 1) / warps;
  if (blocks > c->num_sms) blocks = c->num_sms;
  const size_t smem = (smem_tables ? table_bytes : 0) + priv_per_warp * warps;
  if (smem_tables) {
    cudaFuncSetAttribute(whp_legs_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
    whp_legs_kernel<true, false><<<(unsigned)blocks, warps * 32, smem, st>>>(
        T, P, c->d_pick_fast, c->d_cstream, c->d_bmask, c->d_nb, c->d_segstart, n_cand, d_len, c->d_task);
  } else if (fours) {
    cudaFuncSetAttribute(whp_legs_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
    whp_legs_kernel<false, true><<<(unsigned)blocks, warps * 32, smem, st>>>(
        T, P, c->d_pick_f4, c->d_cstream, c->d_bmask, c->d_nb, c->d_segstart, n_cand, d_len, c->d_task);
  } else {
    cudaFuncSetAttribute(whp_legs_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
    whp_legs_kernel<false, false><<<(unsigned)blocks, warps * 32, smem, st>>>(
        T, P, c->d_pick_fast, c->d_cstream, c->d_bmask, c->d_nb, c->d_segstart, n_cand, d_len, c->d_task);
  }
  c->launches += 1;
  return cudaGetLastError();
}
