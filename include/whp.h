/* whp.h — C-ABI boundary of the B200-native candidate picking-plan evaluator.
 *
 * What the library computes (one GPU, sm_100a, no collectives):
 *   the data-parallel hot path of subproblem 2 of the paper's NHATC-coordinated warehouse
 *   SDO — "by evaluating the permutations of different picking sequences, can minimum
 *   distance for the picking route be found" (§5 Eq. 2: min Σ d_i), scored
 *   inside an NHATC subproblem  min f_ij(x) + φ(c_ij)  (§5 Eq. 3) where
 *   c is the inconsistency between target t and response r.
 *   The concrete definitions (geometry D0, next-fit batching D2, per-batch sets D3,
 *   S-shape distance D4, responses D5, penalty D6, argmin D7, swap neighbourhood D8) are
 *   the readings listed in DESIGN.md §2 (from SURVEY.md §8(c) and BASELINE.json north_star).
 *
 * Conventions
 *   - Every call returns a whp_status; nothing throws or aborts. whp_last_error() gives text.
 *   - "host" pointers are ordinary CPU memory; they are copied during the call and the
 *     caller keeps ownership. "DEVICE" pointers are caller-owned CUDA device memory on the
 *     ctx's device (e.g. a torch tensor's data_ptr()); the library never frees them.
 *   - eval / argmin / apply calls are asynchronous on `cuda_stream` (a cudaStream_t passed
 *     as void*; NULL = the legacy default stream). Argument errors are detected
 *     synchronously before anything is launched.
 *   - A context owns scratch that its kernels share: calls on one context must not overlap in
 *     time on different streams (serialise them, or use one context per stream). Contexts are
 *     not thread-safe; different contexts are independent.
 *   - CUDA graphs: scratch grows on the first call that needs more of it (that call allocates
 *     and synchronises the stream). Once every call of a loop has run once at its sizes, the
 *     calls that take a `cuda_stream` neither allocate nor synchronise and may be captured
 *     (cudaStreamBeginCapture ... EndCapture) and replayed; scalar arguments such as win_start
 *     are baked into the captured launches. Calls that hand a value back to the host
 *     (the *_host entry points, whp_validate_perms, whp_get_penalty, whp_get_swap_stats,
 *     whp_probe_l2_read)
 *     synchronise and cannot be captured.
 *   - All arrays are dense, row-major, native-endian.
 *   - A row of d_perms that is not a permutation of 0..n_orders-1 is a precondition
 *     violation (entries outside [0,n_orders) would read out of bounds); use
 *     whp_validate_perms when the source is untrusted.
 *
 * Limits (WHP_ERR_OUT_OF_RANGE beyond them): n_aisles <= 1024, slots_per_side <= 4095,
 *   n_classes <= 256, n_orders < 2^24, total items < 2^24, cart_capacity < 2^20, at most 255
 *   items per order.
 *   The tuned kernels additionally need n_orders < 65536, cart_capacity <= 106 and pick cursors
 *   that fit 16 bits; other shapes run the general (slower) kernels with
 *   the same results.
 */
#ifndef WHP_H
#define WHP_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct whp_ctx whp_ctx; /* opaque; owns packed device tables and scratch */

typedef enum {
  WHP_OK = 0,
  WHP_ERR_INVALID_ARG = 1,  /* null pointer, non-positive size, K < 1, W < 2 ...          */
  WHP_ERR_OUT_OF_RANGE = 2, /* loc / sku / class / window outside bounds; non-finite t,v,w;
                               a documented limit exceeded                                  */
  WHP_ERR_CAPACITY = 3,     /* some order has more items than cart_capacity               */
  WHP_ERR_STATE = 4,        /* eval before whp_load_orders / whp_set_penalty              */
  WHP_ERR_CUDA = 5,         /* a CUDA runtime call failed (text in whp_last_error)        */
  WHP_ERR_NOMEM = 6
} whp_status;

/* D0 geometry + SKU tables (BASELINE.json north_star: "whp_create_layout (aisles, slots,
 * SKU→location assignment from category clustering)").
 *   Location l in [0, 2*n_aisles*slots_per_side): aisle = l / (2S), slot = l % S,
 *   depth = (slot+1)*slot_pitch; aisle length A = (S+1)*slot_pitch; aisle a at x = a*aisle_spacing;
 *   depot at the front of depot_aisle.
 *   sku_loc   host int32[n_skus]  location of each SKU
 *   sku_class host int32[n_skus]  workload class (category x zone) in [0, n_classes)
 *   cuda_device: ordinal; *out receives the new context. */
whp_status whp_create_layout(int32_t n_aisles, int32_t slots_per_side, int32_t slot_pitch,
                             int32_t aisle_spacing, int32_t depot_aisle, int32_t n_skus,
                             const int32_t* sku_loc, const int32_t* sku_class,
                             int32_t n_classes, int32_t cuda_device, whp_ctx** out);

/* D1 orders in CSR form. order_ptr host int32[n_orders+1], strictly increasing from 0;
 * item_sku host int32[order_ptr[n_orders]] (an order may repeat a SKU, each repeat is one
 * item). Every order must satisfy q_o <= cart_capacity (else WHP_ERR_CAPACITY, reading Q5).
 * Packs the per-order and per-pick device tables; may be called again to replace them. */
whp_status whp_load_orders(whp_ctx* ctx, int32_t n_orders, const int32_t* order_ptr,
                           const int32_t* item_sku, int32_t cart_capacity);

/* D6 penalty parameters: targets t, multipliers v, weights w; host double[n_classes] each,
 * all finite. May be called again (the NHATC outer loop updates them). */
whp_status whp_set_penalty(whp_ctx* ctx, const double* t, const double* v, const double* w);

/* a1–a5: evaluate n_cand candidate plans. d_perms DEVICE int32[n_cand][n_orders].
 * Outputs, DEVICE, each nullable (a NULL output is simply not written):
 *   d_dist        int64 [n_cand]            D   = Σ_b dist_b              (D4)
 *   d_penalty     double[n_cand]            φ                              (D6)
 *   d_obj         double[n_cand]            J   = (double)D + φ            (D6)
 *   d_n_batches   int32 [n_cand]                                           (D2)
 *   d_batch_hash  uint64[n_cand]            Σ_b (start_pos_b+1)(2b+1) mod 2^64 (D2)
 *   d_batch_of_pos int32[n_cand][n_orders]  batch index of every position  (D2)
 *   d_n_distinct  int32 [n_cand]            Σ_b |distinct locations of b|  (D3)
 *   d_resp        int32 [n_cand][n_classes] r_k                            (D5)
 * n_cand == 0 is a no-op returning WHP_OK. */
whp_status whp_eval_candidates(whp_ctx* ctx, const int32_t* d_perms, int64_t n_cand,
                               int64_t* d_dist, double* d_penalty, double* d_obj,
                               int32_t* d_n_batches, uint64_t* d_batch_hash,
                               int32_t* d_batch_of_pos, int32_t* d_n_distinct,
                               int32_t* d_resp, void* cuda_stream);

/* Same computation through HOST buffers (the end-to-end path): h_perms host
 * int32[n_cand][n_orders]; h_dist / h_obj host arrays [n_cand] (nullable). Permutations are
 * copied to the device in chunks overlapped with evaluation; results are copied back; the
 * call returns after everything has completed. Pinned host memory makes the copies
 * asynchronous, pageable memory works but serialises. The call runs on streams of its own and
 * does not order itself after work the caller queued earlier on this context (e.g. a
 * whp_nhatc_update still in flight): the context must be idle when it is called. */
whp_status whp_eval_candidates_host(whp_ctx* ctx, const int32_t* h_perms, int64_t n_cand,
                                    int64_t* h_dist, double* h_obj,
                                    int64_t* h_argmin_idx, double* h_argmin_val);

/* The same with 16-bit order ids (h_perms host uint16[n_cand][n_orders]): half the bytes over
 * PCIe, which is what bounds the host-buffer path; the first kernel reads 16-bit tiles. Legal only
 * on shapes of the tuned kernels (n_orders < 65536, ...: WHP_ERR_OUT_OF_RANGE otherwise — use the
 * int32 call). PAPER.md:125 ("evaluating the permutations of different picking sequences");
 * BASELINE.json configs[3] states int32 ids, so the int32 call stays the reference entry point. */
whp_status whp_eval_candidates_host16(whp_ctx* ctx, const uint16_t* h_perms, int64_t n_cand,
                                      int64_t* h_dist, double* h_obj,
                                      int64_t* h_argmin_idx, double* h_argmin_val);

/* a6 (D8): all W(W-1)/2 pairwise swaps of positions inside [win_start, win_start+win_len)
 * of d_base_perm (DEVICE int32[n_orders]); neighbour n <-> (i',j'), 0 <= i' < j' < W,
 * n = i'(2W-i'-1)/2 + (j'-i'-1); value = D2–D6 of the swapped sequence. Only the batches a
 * swap can affect are rescored. d_dist int64 / d_obj double DEVICE [W(W-1)/2], nullable. */
whp_status whp_eval_swaps(whp_ctx* ctx, const int32_t* d_base_perm, int32_t win_start,
                          int32_t win_len, int64_t* d_dist, double* d_obj, void* cuda_stream);

/* a7 (D7): index of the minimum of d_obj[0..n), ties -> lowest index. d_idx int64*, d_val
 * double* are DEVICE scalars (d_val nullable). n must be >= 1. */
whp_status whp_argmin(whp_ctx* ctx, const double* d_obj, int64_t n, int64_t* d_idx,
                      double* d_val, void* cuda_stream);

/* a7 (D7) again, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): the ONE entry point that allocates nothing — no
 * context (creating one allocates), no cudaMalloc / cudaFree / allocating library routine, only a
 * 4-byte cudaMemsetAsync and one kernel on cuda_stream of the CURRENT device. Same result as
 * whp_argmin: *d_idx = index of the minimum of d_obj[0..n) (DEVICE double), ties -> lowest
 * index; *d_val (nullable) its value. d_idx int64*, d_val double* are DEVICE scalars.
 *   - The per-block partial results live in a static __device__ array of
 *     WHP_ARGMIN_STATIC_SCRATCH_BYTES that every GPU loading the library holds until exit; it has
 *     room for 4096 blocks of 4096 values, so n <= WHP_ARGMIN_STATIC_MAX_N. A larger n returns
 *     WHP_ERR_OUT_OF_RANGE (nothing is launched; use whp_argmin); n < 1 or a null d_obj / d_idx
 *     WHP_ERR_INVALID_ARG; a failing CUDA call WHP_ERR_CUDA. Text: whp_static_last_error().
 *   - ALL calls on a device share that array. Calls ordered on one stream (or otherwise
 *     serialised) are fine — the array is re-initialised by every call; calls that OVERLAP on the
 *     GPU (different streams, no dependency) race on it and return garbage.
 *   - whp_argmin_static_setup() resolves the array's device address for the current device
 *     (cudaGetSymbolAddress, once per device). whp_argmin_static does the same on its first call
 *     per device; call the set-up beforehand when that first call would fall inside a stream
 *     capture. Device ordinals 0..63. */
#define WHP_ARGMIN_STATIC_MAX_N 16777216LL      /* 4096 blocks x 4096 values */
#define WHP_ARGMIN_STATIC_SCRATCH_BYTES 65792   /* 4096 x 16 B pairs + a 256 B ticket line */
whp_status whp_argmin_static_setup(void);
whp_status whp_argmin_static(const double* d_obj, int64_t n, int64_t* d_idx, double* d_val,
                             void* cuda_stream);
const char* whp_static_last_error(void); /* of the calling thread's latest *_static call; "" when none */

/* D8 trajectory step: decode neighbour *d_idx (DEVICE int64, as written by whp_argmin over
 * a whp_eval_swaps result with the same window) and exchange the two positions of
 * d_base_perm in place, on the device, so a search loop needs no host round trip. */
whp_status whp_apply_swap(whp_ctx* ctx, int32_t* d_base_perm, int32_t win_start,
                          int32_t win_len, const int64_t* d_idx, void* cuda_stream);

/* ---- NEXT-1: the NHATC outer loop (§5 Eq. 3; update rule = reading N1 of
 * DESIGN.md, the method-of-multipliers step of the cited Tosserams et al. 2010) ------------- */

/* v_k <- v_k + 2 w_k^2 c_k, w_k <- beta w_k with c = t - r*, r* = row *d_idx (DEVICE int64,
 * NULL = row 0) of d_resp_rows (DEVICE int32 [rows][n_classes], e.g. the d_resp output of
 * whp_eval_candidates). Updates the context's penalty parameters in place, on the stream. */
whp_status whp_nhatc_update(whp_ctx* ctx, const int32_t* d_resp_rows, const int64_t* d_idx,
                            double beta, void* cuda_stream);

/* n_outer times { whp_eval_candidates on d_perms -> whp_argmin -> record (winner index, its D,
 * its J) into the DEVICE histories [n_outer] (each nullable) -> whp_nhatc_update with the
 * winner's responses }, all on the stream with no host round trip. The results are those of
 * that loop bit for bit; since D and r of a plan do not depend on (t, v, w), the plans are
 * walked once and the later iterations redo only the penalty (D6) on the stored responses. */
whp_status whp_nhatc_solve(whp_ctx* ctx, const int32_t* d_perms, int64_t n_cand, int32_t n_outer,
                           double beta, int64_t* d_idx_hist, int64_t* d_dist_hist,
                           double* d_obj_hist, void* cuda_stream);

/* Current penalty parameters to HOST double[n_classes] each (nullable). Synchronises the stream. */
whp_status whp_get_penalty(whp_ctx* ctx, double* t, double* v, double* w, void* cuda_stream);

/* ---- NEXT-2: the paper-literal subproblem 2 (§5 Eq. 2: min sum d_i, d_i the
 * shortest-path length between consecutive picking positions; reading N2 of DESIGN.md) ------ */

/* d_len[c] (DEVICE int64 [n_cand]) = summed leg lengths of plan c: every cart (next-fit, D2)
 * leaves the depot, visits its picks in plan order and returns; a leg costs D0's walking
 * metric. d_perms DEVICE int32 [n_cand][n_orders]. Needs whp_load_orders only. */
whp_status whp_eval_legsum(whp_ctx* ctx, const int32_t* d_perms, int64_t n_cand, int64_t* d_len,
                           void* cuda_stream);

/* Routing policies of a cart: the S-shape of D4 (BASELINE.json north_star), and the
 * two further heuristics SURVEY.md §8(f) NEXT-2 names, as read in N5 / N6:
 *   WHP_ROUTE_RETURN       enter every visited aisle from the front cross-aisle, walk to its
 *                          deepest pick and come back: H + 2 * sum over visited aisles of maxdepth
 *   WHP_ROUTE_LARGEST_GAP  one visited aisle: as return; else traverse the first and the last
 *                          visited aisle and enter every aisle in between from the back and / or
 *                          the front so that its largest gap is not walked:
 *                          H + 2A + 2 * sum over inner visited aisles of (A - largest gap)
 * (H = horizontal term of D4, A = aisle length). */
typedef enum {
  WHP_ROUTE_S_SHAPE = 0,
  WHP_ROUTE_RETURN = 1,
  WHP_ROUTE_LARGEST_GAP = 2
} whp_route_policy;

/* D and J = (double)D + phi of every plan with its carts routed by `policy`; batching (D2),
 * responses (D5) and penalty (D6) as in whp_eval_candidates, of which policy 0 is a synonym.
 * d_perms DEVICE int32 [n_cand][n_orders]; d_dist int64 / d_obj double DEVICE [n_cand], nullable.
 * Policies 1 and 2 keep the cart's (aisle, depth) list in shared memory and need
 * cart_capacity <= 1024 (WHP_ERR_OUT_OF_RANGE beyond); an unknown policy is WHP_ERR_INVALID_ARG. */
whp_status whp_eval_routing(whp_ctx* ctx, const int32_t* d_perms, int64_t n_cand, int32_t policy,
                            int64_t* d_dist, double* d_obj, void* cuda_stream);

/* ---- NEXT-3: subproblem 3 (§5: product placement by picking frequency, "e.g.
 * K-means clustering"; reading N3 of DESIGN.md) ------------------------------------------- */

/* K-means (k clusters, `iters` Lloyd iterations + a final assignment) of the n_skus SKUs on
 * their pick frequency in item_sku (host int32 [n_items]), then cluster-contiguous slotting:
 * clusters by centroid (largest first), SKUs by (cluster rank, id), locations by
 * (|aisle - depot_aisle|, aisle, slot, side). Outputs, host: sku_loc, sku_class int32 [n_skus]
 * (class = cluster * n_zones + slot * n_zones / slots_per_side) — the inputs of
 * whp_create_layout with n_classes = k * n_zones; assign int32 [n_skus] and centroids
 * double [k] are nullable. Needs no context; runs on cuda_device and synchronises.
 * Limits: k <= 1024, k * n_zones <= 256, n_skus <= 2 * n_aisles * slots_per_side. */
whp_status whp_kmeans_slotting(int32_t n_aisles, int32_t slots_per_side, int32_t depot_aisle,
                               int32_t n_skus, const int32_t* item_sku, int32_t n_items,
                               int32_t k, int32_t n_zones, int32_t iters, int32_t cuda_device,
                               int32_t* sku_loc, int32_t* sku_class, int32_t* assign,
                               double* centroids);

/* ---- NEXT-4: insertion (or-opt, one order) neighbourhood on the incremental evaluator
 * (reading N4 of DESIGN.md) ------------------------------------------------ */

/* All W(W-1) moves inside [win_start, win_start+win_len) of d_base_perm (DEVICE int32
 * [n_orders]): move (i', j'), i' != j', takes the order at position win_start+i' out and puts it
 * back at position win_start+j'; neighbour n = i'(W-1) + (j' < i' ? j' : j'-1); value = D2-D6
 * of the new sequence. d_dist int64 / d_obj double DEVICE [W(W-1)], nullable. */
whp_status whp_eval_moves(whp_ctx* ctx, const int32_t* d_base_perm, int32_t win_start,
                          int32_t win_len, int64_t* d_dist, double* d_obj, void* cuda_stream);

/* Applies move *d_idx (DEVICE int64, as written by whp_argmin over a whp_eval_moves result of
 * the same window) to d_base_perm in place, on the device. */
whp_status whp_apply_move(whp_ctx* ctx, int32_t* d_base_perm, int32_t win_start, int32_t win_len,
                          const int64_t* d_idx, void* cuda_stream);

/* Debug helper: *h_n_bad (host) receives the number of rows of d_perms that are not a
 * permutation of 0..n_orders-1. Synchronises the stream. */
whp_status whp_validate_perms(whp_ctx* ctx, const int32_t* d_perms, int64_t n_cand,
                              int64_t* h_n_bad, void* cuda_stream);

/* Debug / measurement switch on the kernel selection of ONE context (the results never change,
 * only which kernels compute them; tests use it to reach every code path). value < 0 restores the
 * default. Takes effect from the next call on the context; not meant for production use.
 *   WHP_DEBUG_FORCE_GENERAL  value != 0: whp_eval_candidates / whp_eval_legsum / whp_eval_routing
 *                            take the general warp-per-plan kernels even on tuned-path shapes
 *   WHP_DEBUG_SEGMENTS       segments per plan of the tuned path (a power of two <= 32; ignored
 *                            when the plan's batch count does not allow it)
 *   WHP_DEBUG_WARPS          warps per block of the tuned set kernel (capped by what fits)
 *   WHP_DEBUG_SWAP_MARGIN    positions after the window that whp_eval_swaps / whp_eval_moves
 *                            tabulate (0 forces the batch-by-batch fallback of every chain)
 *   WHP_DEBUG_K1_WARPS       warps per block of the tuned boundary kernel (1, 2, 4 or 5: they share
 *                            one copy of the order table; ignored when it does not fit)
 *   WHP_DEBUG_NO_FOURS       value != 0: pick tables that do not fit shared memory are read by the
 *                            pair-load variant of the set kernel instead of the four-aligned one
 * Unknown keys return WHP_ERR_INVALID_ARG. There are no environment variables. */
typedef enum {
  WHP_DEBUG_FORCE_GENERAL = 0,
  WHP_DEBUG_SEGMENTS = 1,
  WHP_DEBUG_WARPS = 2,
  WHP_DEBUG_SWAP_MARGIN = 3,
  WHP_DEBUG_K1_WARPS = 4,
  WHP_DEBUG_NO_FOURS = 5
} whp_debug_key;
whp_status whp_debug_set(whp_ctx* ctx, int32_t key, int64_t value);

/* Measurement helper ("actually-rescored picks"): with enable != 0 every later
 * whp_eval_swaps / whp_eval_moves call also counts the batches it scored from their picks and
 * the picks in them (everything else in a neighbour's value is table look-ups); off by default.
 * whp_get_swap_stats copies the counts of the latest such call to the host (each nullable) and
 * synchronises the stream. */
whp_status whp_set_swap_stats(whp_ctx* ctx, int32_t enable);
whp_status whp_get_swap_stats(whp_ctx* ctx, int64_t* h_batches, int64_t* h_picks,
                              void* cuda_stream);

/* Measurement helper (bench.py): *h_ms (host) = time of `reps` read-only sweeps (16-byte loads
 * that bypass L1) of a `bytes`-sized buffer, which stays L2-resident when bytes is well below the
 * L2 size. Allocates and frees its own buffer; synchronises. */
whp_status whp_probe_l2_read(whp_ctx* ctx, int64_t bytes, int32_t reps, float* h_ms);

/* Upper bound on the number of carts of ANY plan over the loaded orders (0 before
 * whp_load_orders): the first orders of carts 1..nb-1 are distinct and each did not fit, so
 * (nb-1)(C+1) - (sum of the nb-1 largest item counts) <= n_items - 1. The tuned kernels size
 * their per-segment counters with it. */
int64_t whp_max_batches(const whp_ctx* ctx);

/* Kernel launches issued by this ctx since creation (bench.py's gpu_launches claim). */
int64_t whp_launch_count(const whp_ctx* ctx);

void whp_destroy(whp_ctx* ctx);
const char* whp_last_error(const whp_ctx* ctx); /* "" when none; valid until next call */
const char* whp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WHP_H */
