// whp_internal.cuh — context, packed table formats and launch prototypes shared by the .cu
// files of libwhp.so. Not part of the public boundary (include/whp.h is).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/whp.h"

// ---- packed device tables -----------------------------------------------------
// order record, 32 bit:  item_off[31:8] | q[7:0]            (q = number of items, 1..255)
// pick  record, 32 bit:  0 [31] | aisle[30:21] | slot1[20:9] | side[8] | class[7:0]
//   slot1 = slot + 1 (depth = slot1 * slot_pitch). The field order makes an unsigned max (min)
//   over the records of a batch return (a_max, deepest slot in a_max) ((a_min, ..)) in its top
//   bits (D3). rec >> 26 is the index of the 32-aisle occupancy word and (rec >> 21) mod 32 the
//   bit inside it; (rec & 0xe0) >> 5 the 32-class word and rec mod 32 the bit — so a funnel
//   shift that wraps its shift amount needs no mask.
#define WHP_Q_BITS 8
#define WHP_Q_MASK 0xffu
#define WHP_PICK_PACK_AISLE(a) ((uint32_t)(a) << 21)
#define WHP_PICK_AISLE(rec) ((rec) >> 21)
#define WHP_PICK_SLOT_SHIFT 9
#define WHP_PICK_SLOT_MASK 0xfffu
#define WHP_PICK_LOC_SHIFT 8 /* rec >> 8 identifies the location (aisle, slot, side) */
#define WHP_PICK_CLASS_MASK 0xffu

// pick record of the tuned candidate path (whp_fast.cu), built from the record above:
//   aisle[31:22] | slot1[21:10] | class>>5 [9:7] | last-four [6] | last-pick-of-its-order [5] | class&31 [4:0]
//   (rec >> 20) & (words-1)<<7 and rec & 0x380 are the byte offsets of the 32-aisle and the
//   32-class occupancy words of a lane; (rec >> 22) mod 32 and rec mod 32 the bits inside them.
#define WHP_FAST_LAST 0x20u
#define WHP_FAST_LAST4 0x40u /* four-aligned layout: last record of the order's last four */
#define WHP_FAST_PACK(rec, last)                                                              \
  ((WHP_PICK_AISLE(rec) << 22) | ((((rec) >> WHP_PICK_SLOT_SHIFT) & WHP_PICK_SLOT_MASK) << 10) | \
   ((((rec) & WHP_PICK_CLASS_MASK) >> 5) << 7) | ((last) ? WHP_FAST_LAST : 0u) | ((rec) & 31u))
#define WHP_FAST_AISLE(rec) ((rec) >> 22)
#define WHP_FAST_SLOT1(rec) (((rec) >> 10) & 0xfffu)

#define WHP_MAX_AISLES 1024
#define WHP_MAX_SLOTS 4095
#define WHP_MAX_CLASSES 256
#define WHP_MAX_ITEMS (1 << 24)
#define WHP_MAX_ORDER_ITEMS 255

struct whp_geom {
  int32_t n_aisles, slots_per_side, slot_pitch, aisle_spacing, depot_aisle;
  int64_t aisle_len;  // A = (S+1)*p
};

// Read-only view of everything a kernel needs (passed by value).
struct whp_tables {
  whp_geom g;
  int32_t n_orders, n_items, C, K;
  const uint32_t* order_rec;  // [n_orders]
  const uint32_t* pick_rec;   // [n_items]
  const double* tvw;          // [3][K]: t, v, w
};

// Per-plan outputs of the candidate walker; any pointer may be null.
struct whp_eval_out {
  int64_t* dist;
  double* penalty;
  double* obj;
  int32_t* n_batches;
  uint64_t* batch_hash;
  int32_t* batch_of_pos;
  int32_t* n_distinct;
  int32_t* resp;
};

// Per-batch tables of the base plan, produced by the base pass of whp_eval_swaps (scratch).
struct whp_base_tables {
  int32_t* bstart;    // [n_orders+1] first position of batch b; bstart[nb] = n_orders
  int32_t* bop;       // [n_orders]   batch of position
  int64_t* bdist;     // [n_orders+1] exclusive prefix sum of per-batch S-shape lengths
  int32_t* resp;      // [K]          base responses
  int64_t* totals;    // [2]          D_base, n_batches
  int32_t* pre;       // [n_orders+1] exclusive prefix of the item counts along the plan
  uint32_t* orec;     // [n_orders]   order record of every position
  int32_t* rpre;      // [nb_max+1][K] class-visit counts of the batches before b
  int32_t* nxt;       // [n_orders]   end of the batch that would open at position p
  int64_t* dist_at;   // [n_orders]   S-shape length of that batch (region of the window only)
  uint32_t* cls_at;   // [n_orders][8] its class mask
  int64_t* dtail;     // [n_orders]   chain sums (whp_swaps_chain_kernel), region only
  int32_t* bF;        // [n_orders]   base batch where the chain of p meets the base plan
  int32_t* rtail;     // [region][K]  class visits along the chain
};

struct whp_ctx {
  int device = 0;
  whp_geom g{};
  int32_t n_skus = 0, K = 0;
  int32_t* h_sku_loc = nullptr;  // host copies (needed again by whp_load_orders)
  int32_t* h_sku_class = nullptr;
  // orders
  int32_t n_orders = 0, n_items = 0, C = 0;
  int64_t nb_ub = 0;  // upper bound on the number of batches of ANY plan (whp_load_orders)
  uint32_t* d_order_rec = nullptr;
  uint32_t* d_pick_rec = nullptr;
  // tuned-path tables: every order's picks start at an even index (one pad word after an odd
  // order), bit 8 = "last pick of its order"; order_fast = (first_pick_index/2) << 8 | q
  uint32_t* d_pick_fast = nullptr;
  uint32_t* d_order_fast = nullptr;
  int32_t n_items_pad = 0;
  bool fast_tables_ok = false;
  // second layout for pick tables that do not fit shared memory (K2 gathers them through L1 / L2,
  // whp_sets4_kernel): every order's picks start at a multiple of FOUR and are padded to a
  // multiple of four by repeating the order's last record (set inserts and max are idempotent);
  // the last record of an order's last four carries WHP_FAST_LAST4;
  // order_fast4 = (first_pick_index/4) << 8 | q. Null when the pair table is small or the
  // four-cursors overflow 16 bits.
  uint32_t* d_pick_f4 = nullptr;
  uint32_t* d_order_fast4 = nullptr;
  double* d_tvw = nullptr;
  bool have_orders = false, have_penalty = false;
  // scratch
  whp_base_tables base{};
  int64_t rtail_rows = 0;
  void* d_argmin_part = nullptr;  // partial (val, idx) pairs + ticket
  int32_t argmin_cap = 0;
  unsigned long long* d_count = nullptr;  // validate_perms counter
  // fast candidate path scratch (whp_fast.cu), grow-only
  uint32_t* d_bmask = nullptr;       // [fast_cap][fast_pitch] bitmask of batch-start positions
  uint16_t* d_cstream = nullptr;     // [fast_cap][cs_pitch] first-pick cursor of every position
  int32_t* d_nb = nullptr;           // [fast_cap]
  int32_t* d_segstart = nullptr;     // [fast_cap][32] first position of every segment
  int32_t* d_perm_pad = nullptr;     // padded copy of the plans (n_orders % 4 != 0 or unaligned)
  size_t perm_pad_bytes = 0;
  int64_t* d_dist_scratch = nullptr; // [fast_cap]
  uint32_t* d_planes = nullptr;      // [fast_cap][S][8 planes][KW] bit-sliced class counters
  unsigned long long* d_task = nullptr;  // [2] work-stealing counter
  unsigned long long* d_swap_stats = nullptr;  // [2] batches / picks scored from their picks
  bool swap_stats = false;                     // whp_set_swap_stats
  int64_t fast_cap = 0, fast_plane_words = 0;
  int32_t fast_pitch = 0;
  int smem_optin = 0;
  // host-path staging (whp_eval_candidates_host)
  void* d_stage[2] = {nullptr, nullptr};
  int64_t stage_bytes = 0;
  int64_t* d_h_dist = nullptr;
  double* d_h_obj = nullptr;
  int64_t h_out_cap = 0;
  int64_t* d_h_idx = nullptr;
  // NHATC outer loop scratch (whp_nhatc_solve), grow-only
  int32_t* d_n_resp = nullptr;  // [n_cand][K]
  int64_t n_resp_cap = 0;
  double* d_h_val = nullptr;
  cudaStream_t s_copy[2] = {nullptr, nullptr};
  cudaStream_t s_exec = nullptr;
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr};
  std::vector<cudaEvent_t> ev_piece;  // one per staged piece of whp_eval_candidates_host
  int num_sms = 148;
  int64_t launches = 0;
  // whp_debug_set: kernel-selection overrides for tests and measurements (-1 / 0 = default)
  int32_t dbg_force_general = 0, dbg_segments = -1, dbg_warps = -1, dbg_k1_warps = -1, dbg_no_fours = 0;
  int64_t dbg_swap_margin = -1;
  std::string err;
};

whp_tables whp_make_tables(const whp_ctx* c);

// kernels' host launchers (each returns the cudaError_t of the launch)
cudaError_t whp_launch_eval(whp_ctx* c, const int32_t* d_perms, int64_t n_cand,
                            const whp_eval_out& out, cudaStream_t st);
bool whp_fast_eligible(const whp_ctx* c);
// perm16: d_perms holds uint16 order ids (tuned path only)
cudaError_t whp_launch_eval_fast(whp_ctx* c, const void* d_perms, int64_t n_cand,
                                 const whp_eval_out& out, cudaStream_t st, bool perm16 = false);
cudaError_t whp_launch_swaps(whp_ctx* c, const int32_t* d_base_perm, int32_t win_start,
                             int32_t win_len, int64_t* d_dist, double* d_obj, cudaStream_t st);
cudaError_t whp_launch_moves(whp_ctx* c, const int32_t* d_base_perm, int32_t win_start,
                             int32_t win_len, int64_t* d_dist, double* d_obj, cudaStream_t st);
cudaError_t whp_launch_apply_move(whp_ctx* c, int32_t* d_base_perm, int32_t win_start,
                                  int32_t win_len, const int64_t* d_idx, cudaStream_t st);
cudaError_t whp_launch_argmin(whp_ctx* c, const double* d_obj, int64_t n, int64_t* d_idx,
                              double* d_val, cudaStream_t st);
cudaError_t whp_launch_apply_swap(whp_ctx* c, int32_t* d_base_perm, int32_t win_start,
                                  int32_t win_len, const int64_t* d_idx, cudaStream_t st);
cudaError_t whp_launch_nhatc_update(whp_ctx* c, const int32_t* d_resp_rows, const int64_t* d_idx,
                                    double beta, cudaStream_t st);
cudaError_t whp_launch_nhatc_rescore(whp_ctx* c, const int32_t* d_resp_rows, const int64_t* d_dist,
                                     int64_t n_cand, double* d_obj, cudaStream_t st);
cudaError_t whp_launch_nhatc_record(whp_ctx* c, const int64_t* d_idx, const int64_t* dist,
                                    const double* obj, int32_t it, int64_t* idx_hist,
                                    int64_t* dist_hist, double* obj_hist, cudaStream_t st);
cudaError_t whp_launch_legsum_fast(whp_ctx* c, const int32_t* d_perms, int64_t n_cand, int64_t* d_len,
                                   cudaStream_t st);
cudaError_t whp_launch_legsum(whp_ctx* c, const int32_t* d_perms, int64_t n_cand, int64_t* d_len,
                              cudaStream_t st);
cudaError_t whp_launch_route(whp_ctx* c, const int32_t* d_perms, int64_t n_cand, int32_t policy,
                             int64_t* d_dist, double* d_obj, cudaStream_t st);
cudaError_t whp_launch_l2_probe(whp_ctx* c, int64_t bytes, int32_t reps, float* ms);
cudaError_t whp_launch_validate(whp_ctx* c, const int32_t* d_perms, int64_t n_cand,
                                cudaStream_t st);
