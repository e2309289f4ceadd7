// whp_api.cu — the extern "C" boundary (include/whp.h): argument checking, table packing,
// device memory owned by the context, and dispatch to the kernel launchers. No arithmetic of
// the method happens on the host: the host only validates and packs inputs.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <algorithm>
#include <vector>

#include <nvtx3/nvToolsExt.h>  // header-only: ranges cost nothing unless a profiler is attached

#include "whp_internal.cuh"

namespace {

// NVTX range around an entry point (the layout "is chosen to evaluate
// possible bottlenecks in a specific subprocess"): nsys / ncu --nvtx show the calls by name.
struct nvtx_range {
  explicit nvtx_range(const char* name) { nvtxRangePushA(name); }
  ~nvtx_range() { nvtxRangePop(); }
};

whp_status fail(whp_ctx* c, whp_status s, const char* msg) {
  if (c) c->err = msg;
  return s;
}
whp_status cuda_fail(whp_ctx* c, cudaError_t e, const char* where) {
  if (c) c->err = std::string(where) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? WHP_ERR_NOMEM : WHP_ERR_CUDA;
}
#define WHP_CUDA(c, call)                                        \
  do {                                                           \
    cudaError_t e_ = (call);                                     \
    if (e_ != cudaSuccess) return cuda_fail((c), e_, #call);     \
  } while (0)

struct device_guard {
  int prev = -1;
  explicit device_guard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
  ~device_guard() { if (prev >= 0) cudaSetDevice(prev); }
};

template <class T>
void dfree(T*& p) { if (p) { cudaFree(p); p = nullptr; } }

void free_orders(whp_ctx* c) {
  dfree(c->d_order_rec); dfree(c->d_pick_rec); dfree(c->d_pick_fast); dfree(c->d_order_fast);
  dfree(c->d_pick_f4); dfree(c->d_order_fast4);
  dfree(c->base.bstart); dfree(c->base.bop); dfree(c->base.bdist);
  dfree(c->base.resp); dfree(c->base.totals); dfree(c->base.pre);
  dfree(c->base.orec); dfree(c->base.rpre); dfree(c->base.nxt); dfree(c->base.dist_at);
  dfree(c->base.cls_at); dfree(c->base.dtail); dfree(c->base.bF); dfree(c->base.rtail);
  c->rtail_rows = 0;
  dfree(c->d_stage[0]); dfree(c->d_stage[1]);
  c->stage_bytes = 0;
  dfree(c->d_bmask); dfree(c->d_cstream); dfree(c->d_nb); dfree(c->d_dist_scratch);
  dfree(c->d_planes); dfree(c->d_segstart); dfree(c->d_perm_pad);
  c->perm_pad_bytes = 0;
  c->fast_cap = 0; c->fast_pitch = 0; c->fast_plane_words = 0;
  c->have_orders = false;
}

}  // namespace

whp_tables whp_make_tables(const whp_ctx* c) {
  whp_tables T;
  T.g = c->g;
  T.n_orders = c->n_orders; T.n_items = c->n_items; T.C = c->C; T.K = c->K;
  T.order_rec = c->d_order_rec; T.pick_rec = c->d_pick_rec; T.tvw = c->d_tvw;
  return T;
}

extern "C" {

const char* whp_version(void) { return "whp 0.1 (sm_100a)"; }

const char* whp_last_error(const whp_ctx* c) { return c ? c->err.c_str() : "null context"; }

int64_t whp_launch_count(const whp_ctx* c) { return c ? c->launches : 0; }

int64_t whp_max_batches(const whp_ctx* c) { return (c && c->have_orders) ? c->nb_ub : 0; }

whp_status whp_create_layout(int32_t n_aisles, int32_t slots_per_side, int32_t slot_pitch,
                             int32_t aisle_spacing, int32_t depot_aisle, int32_t n_skus,
                             const int32_t* sku_loc, const int32_t* sku_class, int32_t n_classes,
                             int32_t cuda_device, whp_ctx** out) {
  nvtx_range nvtx_("whp_create_layout");
  if (!out) return WHP_ERR_INVALID_ARG;
  *out = nullptr;
  if (!sku_loc || !sku_class) return WHP_ERR_INVALID_ARG;
  if (n_aisles < 1 || slots_per_side < 1 || slot_pitch < 1 || aisle_spacing < 1 || n_skus < 1 ||
      n_classes < 1 || cuda_device < 0)
    return WHP_ERR_INVALID_ARG;
  if (n_aisles > WHP_MAX_AISLES || slots_per_side > WHP_MAX_SLOTS ||
      n_classes > WHP_MAX_CLASSES || depot_aisle < 0 || depot_aisle >= n_aisles)
    return WHP_ERR_OUT_OF_RANGE;
  const int64_t n_loc = 2ll * n_aisles * slots_per_side;
  for (int32_t s = 0; s < n_skus; ++s) {
    if (sku_loc[s] < 0 || sku_loc[s] >= n_loc) return WHP_ERR_OUT_OF_RANGE;
    if (sku_class[s] < 0 || sku_class[s] >= n_classes) return WHP_ERR_OUT_OF_RANGE;
  }
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cuda_device >= n_dev) return WHP_ERR_CUDA;
  whp_ctx* c = new (std::nothrow) whp_ctx();
  if (!c) return WHP_ERR_NOMEM;
  c->device = cuda_device;
  c->g.n_aisles = n_aisles; c->g.slots_per_side = slots_per_side; c->g.slot_pitch = slot_pitch;
  c->g.aisle_spacing = aisle_spacing; c->g.depot_aisle = depot_aisle;
  c->g.aisle_len = (int64_t)(slots_per_side + 1) * slot_pitch;
  c->n_skus = n_skus; c->K = n_classes;
  c->h_sku_loc = (int32_t*)malloc(sizeof(int32_t) * (size_t)n_skus);
  c->h_sku_class = (int32_t*)malloc(sizeof(int32_t) * (size_t)n_skus);
  if (!c->h_sku_loc || !c->h_sku_class) { whp_destroy(c); return WHP_ERR_NOMEM; }
  memcpy(c->h_sku_loc, sku_loc, sizeof(int32_t) * (size_t)n_skus);
  memcpy(c->h_sku_class, sku_class, sizeof(int32_t) * (size_t)n_skus);
  device_guard dg(cuda_device);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) { whp_destroy(c); return WHP_ERR_CUDA; }
  c->num_sms = prop.multiProcessorCount;
  c->argmin_cap = c->num_sms * 4;
  c->smem_optin = (int)prop.sharedMemPerBlockOptin;
  cudaError_t e = cudaMalloc(&c->d_tvw, sizeof(double) * 3 * (size_t)n_classes);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_argmin_part, 16 * (size_t)c->argmin_cap + 16);
  if (e == cudaSuccess) e = cudaMemset(c->d_argmin_part, 0, 16 * (size_t)c->argmin_cap + 16);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_count, sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMalloc(&c->d_task, 2 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMalloc(&c->d_swap_stats, 2 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMemset(c->d_swap_stats, 0, 2 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMalloc(&c->d_h_idx, sizeof(int64_t));
  if (e == cudaSuccess) e = cudaMalloc(&c->d_h_val, sizeof(double));
  for (int k = 0; k < 2 && e == cudaSuccess; ++k) {
    e = cudaStreamCreateWithFlags(&c->s_copy[k], cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_copied[k], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_done[k], cudaEventDisableTiming);
  }
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->s_exec, cudaStreamNonBlocking);
  if (e != cudaSuccess) { whp_status s = e == cudaErrorMemoryAllocation ? WHP_ERR_NOMEM : WHP_ERR_CUDA; whp_destroy(c); return s; }
  *out = c;
  return WHP_OK;
}

whp_status whp_load_orders(whp_ctx* c, int32_t n_orders, const int32_t* order_ptr,
                           const int32_t* item_sku, int32_t cart_capacity) {
  nvtx_range nvtx_("whp_load_orders");
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  if (!order_ptr || !item_sku || n_orders < 1 || cart_capacity < 1)
    return fail(c, WHP_ERR_INVALID_ARG, "null pointer or non-positive size");
  if (n_orders >= (1 << 24) || cart_capacity >= (1 << 20))
    return fail(c, WHP_ERR_OUT_OF_RANGE, "n_orders or cart_capacity beyond the documented limit");
  if (order_ptr[0] != 0) return fail(c, WHP_ERR_INVALID_ARG, "order_ptr[0] must be 0");
  for (int32_t o = 0; o < n_orders; ++o) {
    const int64_t q = (int64_t)order_ptr[o + 1] - order_ptr[o];
    if (q < 1) return fail(c, WHP_ERR_INVALID_ARG, "order_ptr must be strictly increasing");
    if (q > cart_capacity) return fail(c, WHP_ERR_CAPACITY, "an order exceeds the cart capacity");
    if (q > WHP_MAX_ORDER_ITEMS) return fail(c, WHP_ERR_OUT_OF_RANGE, "an order has more than 255 items");
  }
  const int32_t n_items = order_ptr[n_orders];
  if (n_items >= WHP_MAX_ITEMS) return fail(c, WHP_ERR_OUT_OF_RANGE, "more than 2^24 items");
  for (int32_t i = 0; i < n_items; ++i)
    if (item_sku[i] < 0 || item_sku[i] >= c->n_skus) return fail(c, WHP_ERR_OUT_OF_RANGE, "item_sku out of range");
  // pack (layout in whp_internal.cuh)
  std::vector<uint32_t> orec((size_t)n_orders), prec((size_t)n_items);
  const int32_t S = c->g.slots_per_side;
  for (int32_t o = 0; o < n_orders; ++o)
    orec[o] = ((uint32_t)order_ptr[o] << WHP_Q_BITS) | (uint32_t)(order_ptr[o + 1] - order_ptr[o]);
  for (int32_t i = 0; i < n_items; ++i) {
    const int32_t loc = c->h_sku_loc[item_sku[i]];
    const uint32_t aisle = (uint32_t)(loc / (2 * S)), side = (uint32_t)((loc % (2 * S)) / S);
    const uint32_t slot1 = (uint32_t)(loc % S) + 1u;
    prec[i] = WHP_PICK_PACK_AISLE(aisle) | (slot1 << WHP_PICK_SLOT_SHIFT) |
              (side << WHP_PICK_LOC_SHIFT) | (uint32_t)c->h_sku_class[item_sku[i]];
  }
  device_guard dg(c->device);
  WHP_CUDA(c, cudaDeviceSynchronize());  // nothing may still be reading the old tables
  free_orders(c);
  c->n_orders = n_orders; c->n_items = n_items; c->C = cart_capacity;
  {
    // Upper bound on the batch count of any plan. A cart b closes because the first order f of
    // cart b+1 does not fit: load_b >= C + 1 - q_f. The nb-1 openers are distinct orders, so
    // (nb-1)(C+1) - (sum of the nb-1 largest counts) <= n_items - 1; the left side grows with nb.
    std::vector<int32_t> qs((size_t)n_orders);
    for (int32_t o = 0; o < n_orders; ++o) qs[o] = order_ptr[o + 1] - order_ptr[o];
    std::sort(qs.begin(), qs.end(), [](int32_t a, int32_t b) { return a > b; });
    int64_t m = 0, top = 0;
    while (m < n_orders && (m + 1) * ((int64_t)cart_capacity + 1) - (top + qs[(size_t)m]) <= (int64_t)n_items - 1) {
      top += qs[(size_t)m];
      ++m;
    }
    c->nb_ub = 1 + m < n_orders ? 1 + m : n_orders;
  }
  const size_t no = (size_t)n_orders;
  WHP_CUDA(c, cudaMalloc(&c->d_order_rec, 4 * no));
  WHP_CUDA(c, cudaMalloc(&c->d_pick_rec, 4 * (size_t)n_items));
  WHP_CUDA(c, cudaMalloc(&c->base.bstart, 4 * (no + 1)));
  WHP_CUDA(c, cudaMalloc(&c->base.bop, 4 * no));
  WHP_CUDA(c, cudaMalloc(&c->base.bdist, 8 * (no + 1)));
  WHP_CUDA(c, cudaMalloc(&c->base.resp, 4 * (size_t)c->K));
  WHP_CUDA(c, cudaMalloc(&c->base.totals, 16));
  WHP_CUDA(c, cudaMalloc(&c->base.pre, 4 * (no + 1)));
  WHP_CUDA(c, cudaMalloc(&c->base.orec, 4 * no));
  WHP_CUDA(c, cudaMalloc(&c->base.nxt, 4 * no));
  WHP_CUDA(c, cudaMalloc(&c->base.dist_at, 8 * no));
  WHP_CUDA(c, cudaMalloc(&c->base.cls_at, 32 * no));
  WHP_CUDA(c, cudaMalloc(&c->base.dtail, 8 * no));
  WHP_CUDA(c, cudaMalloc(&c->base.bF, 4 * no));
  {  // consecutive next-fit batches together hold more than C items: nb <= 2 n_items/(C+1) + 1
    int64_t nb_max = 2ll * n_items / ((int64_t)cart_capacity + 1) + 1;
    if (nb_max > n_orders) nb_max = n_orders;
    WHP_CUDA(c, cudaMalloc(&c->base.rpre, 4 * (size_t)(nb_max + 1) * (size_t)c->K));
  }
  WHP_CUDA(c, cudaMemcpy(c->d_order_rec, orec.data(), 4 * no, cudaMemcpyHostToDevice));
  WHP_CUDA(c, cudaMemcpy(c->d_pick_rec, prec.data(), 4 * (size_t)n_items, cudaMemcpyHostToDevice));
  // tuned-path tables (layout in whp_internal.cuh)
  std::vector<uint32_t> ofast((size_t)n_orders), pfast;
  pfast.reserve((size_t)n_items + (size_t)n_orders);
  bool fast_ok = true;
  for (int32_t o = 0; o < n_orders; ++o) {
    const size_t cur = pfast.size() / 2;
    if (cur > 0xffff) fast_ok = false;
    for (int32_t i = order_ptr[o]; i < order_ptr[o + 1]; ++i) {
      const uint32_t r = WHP_FAST_PACK(prec[i], i == order_ptr[o + 1] - 1);
      pfast.push_back(r);
    }
    if (pfast.size() & 1) pfast.push_back(0u);
    ofast[o] = ((uint32_t)(cur & 0xffff) << WHP_Q_BITS) | (uint32_t)(order_ptr[o + 1] - order_ptr[o]);
  }
  c->n_items_pad = (int32_t)pfast.size();
  c->fast_tables_ok = fast_ok;
  WHP_CUDA(c, cudaMalloc(&c->d_pick_fast, 4 * pfast.size()));
  ofast.resize((no + 3) & ~(size_t)3, 0u);  // padded to a multiple of 16 bytes (bulk copy)
  WHP_CUDA(c, cudaMalloc(&c->d_order_fast, 4 * ofast.size()));
  WHP_CUDA(c, cudaMemcpy(c->d_pick_fast, pfast.data(), 4 * pfast.size(), cudaMemcpyHostToDevice));
  WHP_CUDA(c, cudaMemcpy(c->d_order_fast, ofast.data(), 4 * ofast.size(), cudaMemcpyHostToDevice));
  // the four-aligned layout, for tables that cannot sit in shared memory beside K2's private state
  // (built whenever the pair table takes more than half of it; the launch decides which is used)
  if (fast_ok && 4 * pfast.size() > (size_t)c->smem_optin / 2) {
    std::vector<uint32_t> ofast4((no + 3) & ~(size_t)3, 0u), pf4;
    pf4.reserve((size_t)n_items + 3 * (size_t)n_orders);
    bool ok4 = true;
    for (int32_t o = 0; o < n_orders; ++o) {
      const size_t cur = pf4.size() / 4;
      if (cur > 0xffff) { ok4 = false; break; }
      uint32_t r = 0;
      for (int32_t i = order_ptr[o]; i < order_ptr[o + 1]; ++i) {
        r = WHP_FAST_PACK(prec[i], i == order_ptr[o + 1] - 1);
        pf4.push_back(r);
      }
      while (pf4.size() & 3) pf4.push_back(r);  // the order's last record again
      pf4.back() |= WHP_FAST_LAST4;             // this four ends the order
      ofast4[o] = ((uint32_t)cur << WHP_Q_BITS) | (uint32_t)(order_ptr[o + 1] - order_ptr[o]);
    }
    if (ok4) {
      WHP_CUDA(c, cudaMalloc(&c->d_pick_f4, 4 * pf4.size()));
      WHP_CUDA(c, cudaMalloc(&c->d_order_fast4, 4 * ofast4.size()));
      WHP_CUDA(c, cudaMemcpy(c->d_pick_f4, pf4.data(), 4 * pf4.size(), cudaMemcpyHostToDevice));
      WHP_CUDA(c, cudaMemcpy(c->d_order_fast4, ofast4.data(), 4 * ofast4.size(), cudaMemcpyHostToDevice));
    }
  }
  c->have_orders = true;
  return WHP_OK;
}

whp_status whp_set_penalty(whp_ctx* c, const double* t, const double* v, const double* w) {
  nvtx_range nvtx_("whp_set_penalty");
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  if (!t || !v || !w) return fail(c, WHP_ERR_INVALID_ARG, "null pointer");
  std::vector<double> tvw(3 * (size_t)c->K);
  for (int32_t k = 0; k < c->K; ++k) {
    if (!std::isfinite(t[k]) || !std::isfinite(v[k]) || !std::isfinite(w[k]))
      return fail(c, WHP_ERR_OUT_OF_RANGE, "non-finite t, v or w");
    tvw[k] = t[k]; tvw[c->K + k] = v[k]; tvw[2 * (size_t)c->K + k] = w[k];
  }
  device_guard dg(c->device);
  WHP_CUDA(c, cudaDeviceSynchronize());
  WHP_CUDA(c, cudaMemcpy(c->d_tvw, tvw.data(), sizeof(double) * tvw.size(), cudaMemcpyHostToDevice));
  c->have_penalty = true;
  return WHP_OK;
}

static whp_status ready(whp_ctx* c) {
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  if (!c->have_orders) return fail(c, WHP_ERR_STATE, "whp_load_orders has not been called");
  if (!c->have_penalty) return fail(c, WHP_ERR_STATE, "whp_set_penalty has not been called");
  return WHP_OK;
}

whp_status whp_eval_candidates(whp_ctx* c, const int32_t* d_perms, int64_t n_cand,
                               int64_t* d_dist, double* d_penalty, double* d_obj,
                               int32_t* d_n_batches, uint64_t* d_batch_hash,
                               int32_t* d_batch_of_pos, int32_t* d_n_distinct, int32_t* d_resp,
                               void* cuda_stream) {
  nvtx_range nvtx_("whp_eval_candidates");
  whp_status s = ready(c);
  if (s != WHP_OK) return s;
  if (n_cand < 0) return fail(c, WHP_ERR_INVALID_ARG, "n_cand < 0");
  if (n_cand == 0) return WHP_OK;
  if (!d_perms) return fail(c, WHP_ERR_INVALID_ARG, "d_perms is null");
  device_guard dg(c->device);
  whp_eval_out out{d_dist, d_penalty, d_obj, d_n_batches, d_batch_hash, d_batch_of_pos,
                   d_n_distinct, d_resp};
  WHP_CUDA(c, whp_launch_eval(c, d_perms, n_cand, out, (cudaStream_t)cuda_stream));
  return WHP_OK;
}

whp_status whp_eval_swaps(whp_ctx* c, const int32_t* d_base_perm, int32_t win_start,
                          int32_t win_len, int64_t* d_dist, double* d_obj, void* cuda_stream) {
  nvtx_range nvtx_("whp_eval_swaps");
  whp_status s = ready(c);
  if (s != WHP_OK) return s;
  if (!d_base_perm) return fail(c, WHP_ERR_INVALID_ARG, "d_base_perm is null");
  if (win_len < 2) return fail(c, WHP_ERR_INVALID_ARG, "window shorter than 2");
  if (win_start < 0 || (int64_t)win_start + win_len > c->n_orders)
    return fail(c, WHP_ERR_OUT_OF_RANGE, "window outside the plan");
  device_guard dg(c->device);
  WHP_CUDA(c, whp_launch_swaps(c, d_base_perm, win_start, win_len, d_dist, d_obj,
                               (cudaStream_t)cuda_stream));
  return WHP_OK;
}

whp_status whp_argmin(whp_ctx* c, const double* d_obj, int64_t n, int64_t* d_idx, double* d_val,
                      void* cuda_stream) {
  nvtx_range nvtx_("whp_argmin");
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  if (!d_obj || !d_idx || n < 1) return fail(c, WHP_ERR_INVALID_ARG, "null pointer or n < 1");
  device_guard dg(c->device);
  WHP_CUDA(c, whp_launch_argmin(c, d_obj, n, d_idx, d_val, (cudaStream_t)cuda_stream));
  return WHP_OK;
}

whp_status whp_apply_swap(whp_ctx* c, int32_t* d_base_perm, int32_t win_start, int32_t win_len,
                          const int64_t* d_idx, void* cuda_stream) {
  nvtx_range nvtx_("whp_apply_swap");
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  if (!c->have_orders) return fail(c, WHP_ERR_STATE, "whp_load_orders has not been called");
  if (!d_base_perm || !d_idx) return fail(c, WHP_ERR_INVALID_ARG, "null pointer");
  if (win_len < 2) return fail(c, WHP_ERR_INVALID_ARG, "window shorter than 2");
  if (win_start < 0 || (int64_t)win_start + win_len > c->n_orders)
    return fail(c, WHP_ERR_OUT_OF_RANGE, "window outside the plan");
  device_guard dg(c->device);
  WHP_CUDA(c, whp_launch_apply_swap(c, d_base_perm, win_start, win_len, d_idx,
                                    (cudaStream_t)cuda_stream));
  return WHP_OK;
}

whp_status whp_validate_perms(whp_ctx* c, const int32_t* d_perms, int64_t n_cand,
                              int64_t* h_n_bad, void* cuda_stream) {
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  if (!c->have_orders) return fail(c, WHP_ERR_STATE, "whp_load_orders has not been called");
  if (!d_perms || !h_n_bad || n_cand < 0) return fail(c, WHP_ERR_INVALID_ARG, "bad argument");
  *h_n_bad = 0;
  if (n_cand == 0) return WHP_OK;
  if (c->n_orders > (1 << 20)) return fail(c, WHP_ERR_OUT_OF_RANGE, "validate supports n_orders <= 2^20");
  device_guard dg(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  WHP_CUDA(c, cudaMemsetAsync(c->d_count, 0, sizeof(unsigned long long), st));
  WHP_CUDA(c, whp_launch_validate(c, d_perms, n_cand, st));
  unsigned long long bad = 0;
  WHP_CUDA(c, cudaMemcpyAsync(&bad, c->d_count, sizeof(bad), cudaMemcpyDeviceToHost, st));
  WHP_CUDA(c, cudaStreamSynchronize(st));
  *h_n_bad = (int64_t)bad;
  return WHP_OK;
}

// Shared by the two host-buffer entry points: elem = bytes of an order id (4, or 2 for host16).
static whp_status eval_host(whp_ctx* c, const void* h_perms, size_t elem, int64_t n_cand,
                            int64_t* h_dist, double* h_obj, int64_t* h_argmin_idx,
                            double* h_argmin_val) {
  whp_status s = ready(c);
  if (s != WHP_OK) return s;
  if (n_cand < 0) return fail(c, WHP_ERR_INVALID_ARG, "n_cand < 0");
  if (n_cand == 0) return WHP_OK;
  if (!h_perms) return fail(c, WHP_ERR_INVALID_ARG, "h_perms is null");
  const bool perm16 = elem == 2;
  if (perm16 && !whp_fast_eligible(c))
    return fail(c, WHP_ERR_OUT_OF_RANGE, "16-bit plans need a shape of the tuned path (whp.h limits): use whp_eval_candidates_host");
  device_guard dg(c->device);
  // Staging: the plans of one pass (up to 1 GiB of them) go to one device buffer in ~16 MB
  // pieces, ALL enqueued on the copy stream before the first evaluation is launched — the host
  // work of a launch (two tensor-map encodings, four launches) would otherwise sit between two
  // copies and leave PCIe idle. Piece k is evaluated as soon as its copy has landed, so only the
  // last piece's evaluation is not hidden behind a copy.
  const int64_t row_bytes = (int64_t)elem * c->n_orders;
  int64_t rows = (16ll << 20) / row_bytes;
  if (rows < 1) rows = 1;
  int64_t pass_rows = (1ll << 30) / row_bytes;
  if (pass_rows < rows) pass_rows = rows;
  if (pass_rows > n_cand) pass_rows = n_cand;
  if (c->stage_bytes < pass_rows * row_bytes) {
    dfree(c->d_stage[0]);
    c->stage_bytes = 0;
    WHP_CUDA(c, cudaMalloc(&c->d_stage[0], (size_t)(pass_rows * row_bytes)));
    c->stage_bytes = pass_rows * row_bytes;
  }
  const int64_t pieces = (pass_rows + rows - 1) / rows;
  while ((int64_t)c->ev_piece.size() < pieces) {
    cudaEvent_t ev = nullptr;
    WHP_CUDA(c, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    c->ev_piece.push_back(ev);
  }
  if (c->h_out_cap < n_cand) {
    dfree(c->d_h_dist); dfree(c->d_h_obj);
    WHP_CUDA(c, cudaMalloc(&c->d_h_dist, 8 * (size_t)n_cand));
    WHP_CUDA(c, cudaMalloc(&c->d_h_obj, 8 * (size_t)n_cand));
    c->h_out_cap = n_cand;
  }
  for (int64_t pass_lo = 0; pass_lo < n_cand; pass_lo += pass_rows) {
    const int64_t pass_n = (n_cand - pass_lo < pass_rows) ? n_cand - pass_lo : pass_rows;
    if (pass_lo > 0) {  // the buffer is reused: the previous pass must have been evaluated
      WHP_CUDA(c, cudaEventRecord(c->ev_done[0], c->s_exec));
      WHP_CUDA(c, cudaStreamWaitEvent(c->s_copy[0], c->ev_done[0], 0));
    }
    int64_t k = 0;
    for (int64_t lo = 0; lo < pass_n; lo += rows, ++k) {
      const int64_t nr = (pass_n - lo < rows) ? pass_n - lo : rows;
      WHP_CUDA(c, cudaMemcpyAsync((char*)c->d_stage[0] + lo * row_bytes,
                                  (const char*)h_perms + (pass_lo + lo) * row_bytes,
                                  (size_t)(nr * row_bytes), cudaMemcpyHostToDevice, c->s_copy[0]));
      WHP_CUDA(c, cudaEventRecord(c->ev_piece[(size_t)k], c->s_copy[0]));
    }
    k = 0;
    for (int64_t lo = 0; lo < pass_n; lo += rows, ++k) {
      const int64_t nr = (pass_n - lo < rows) ? pass_n - lo : rows;
      WHP_CUDA(c, cudaStreamWaitEvent(c->s_exec, c->ev_piece[(size_t)k], 0));
      whp_eval_out out{c->d_h_dist + pass_lo + lo, nullptr, c->d_h_obj + pass_lo + lo, nullptr,
                       nullptr, nullptr, nullptr, nullptr};
      const void* src = (const char*)c->d_stage[0] + lo * row_bytes;
      if (perm16)
        WHP_CUDA(c, whp_launch_eval_fast(c, src, nr, out, c->s_exec, true));
      else
        WHP_CUDA(c, whp_launch_eval(c, (const int32_t*)src, nr, out, c->s_exec));
    }
  }
  if (h_argmin_idx || h_argmin_val) {
    WHP_CUDA(c, whp_launch_argmin(c, c->d_h_obj, n_cand, c->d_h_idx, c->d_h_val, c->s_exec));
    if (h_argmin_idx)
      WHP_CUDA(c, cudaMemcpyAsync(h_argmin_idx, c->d_h_idx, 8, cudaMemcpyDeviceToHost, c->s_exec));
    if (h_argmin_val)
      WHP_CUDA(c, cudaMemcpyAsync(h_argmin_val, c->d_h_val, 8, cudaMemcpyDeviceToHost, c->s_exec));
  }
  if (h_dist)
    WHP_CUDA(c, cudaMemcpyAsync(h_dist, c->d_h_dist, 8 * (size_t)n_cand, cudaMemcpyDeviceToHost, c->s_exec));
  if (h_obj)
    WHP_CUDA(c, cudaMemcpyAsync(h_obj, c->d_h_obj, 8 * (size_t)n_cand, cudaMemcpyDeviceToHost, c->s_exec));
  WHP_CUDA(c, cudaStreamSynchronize(c->s_exec));
  return WHP_OK;
}

whp_status whp_eval_candidates_host(whp_ctx* c, const int32_t* h_perms, int64_t n_cand,
                                    int64_t* h_dist, double* h_obj, int64_t* h_argmin_idx,
                                    double* h_argmin_val) {
  nvtx_range nvtx_("whp_eval_candidates_host");
  return eval_host(c, h_perms, 4, n_cand, h_dist, h_obj, h_argmin_idx, h_argmin_val);
}

whp_status whp_eval_candidates_host16(whp_ctx* c, const uint16_t* h_perms, int64_t n_cand,
                                      int64_t* h_dist, double* h_obj, int64_t* h_argmin_idx,
                                      double* h_argmin_val) {
  nvtx_range nvtx_("whp_eval_candidates_host16");
  return eval_host(c, h_perms, 2, n_cand, h_dist, h_obj, h_argmin_idx, h_argmin_val);
}

whp_status whp_eval_moves(whp_ctx* c, const int32_t* d_base_perm, int32_t win_start,
                          int32_t win_len, int64_t* d_dist, double* d_obj, void* cuda_stream) {
  nvtx_range nvtx_("whp_eval_moves");
  whp_status s = ready(c);
  if (s != WHP_OK) return s;
  if (!d_base_perm) return fail(c, WHP_ERR_INVALID_ARG, "d_base_perm is null");
  if (win_len < 2) return fail(c, WHP_ERR_INVALID_ARG, "window shorter than 2");
  if (win_start < 0 || (int64_t)win_start + win_len > c->n_orders)
    return fail(c, WHP_ERR_OUT_OF_RANGE, "window outside the plan");
  device_guard dg(c->device);
  WHP_CUDA(c, whp_launch_moves(c, d_base_perm, win_start, win_len, d_dist, d_obj,
                               (cudaStream_t)cuda_stream));
  return WHP_OK;
}

whp_status whp_apply_move(whp_ctx* c, int32_t* d_base_perm, int32_t win_start, int32_t win_len,
                          const int64_t* d_idx, void* cuda_stream) {
  nvtx_range nvtx_("whp_apply_move");
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  if (!c->have_orders) return fail(c, WHP_ERR_STATE, "whp_load_orders has not been called");
  if (!d_base_perm || !d_idx) return fail(c, WHP_ERR_INVALID_ARG, "null pointer");
  if (win_len < 2) return fail(c, WHP_ERR_INVALID_ARG, "window shorter than 2");
  if (win_start < 0 || (int64_t)win_start + win_len > c->n_orders)
    return fail(c, WHP_ERR_OUT_OF_RANGE, "window outside the plan");
  device_guard dg(c->device);
  WHP_CUDA(c, whp_launch_apply_move(c, d_base_perm, win_start, win_len, d_idx,
                                    (cudaStream_t)cuda_stream));
  return WHP_OK;
}

whp_status whp_eval_legsum(whp_ctx* c, const int32_t* d_perms, int64_t n_cand, int64_t* d_len,
                           void* cuda_stream) {
  nvtx_range nvtx_("whp_eval_legsum");
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  if (!c->have_orders) return fail(c, WHP_ERR_STATE, "whp_load_orders has not been called");
  if (n_cand < 0) return fail(c, WHP_ERR_INVALID_ARG, "n_cand < 0");
  if (n_cand == 0) return WHP_OK;
  if (!d_perms || !d_len) return fail(c, WHP_ERR_INVALID_ARG, "null pointer");
  device_guard dg(c->device);
  WHP_CUDA(c, whp_launch_legsum(c, d_perms, n_cand, d_len, (cudaStream_t)cuda_stream));
  return WHP_OK;
}

whp_status whp_eval_routing(whp_ctx* c, const int32_t* d_perms, int64_t n_cand, int32_t policy,
                            int64_t* d_dist, double* d_obj, void* cuda_stream) {
  nvtx_range nvtx_("whp_eval_routing");
  whp_status s = ready(c);
  if (s != WHP_OK) return s;
  if (n_cand < 0) return fail(c, WHP_ERR_INVALID_ARG, "n_cand < 0");
  if (policy < WHP_ROUTE_S_SHAPE || policy > WHP_ROUTE_LARGEST_GAP)
    return fail(c, WHP_ERR_INVALID_ARG, "unknown routing policy");
  if (n_cand == 0) return WHP_OK;
  if (!d_perms) return fail(c, WHP_ERR_INVALID_ARG, "d_perms is null");
  device_guard dg(c->device);
  if (policy == WHP_ROUTE_S_SHAPE) {
    whp_eval_out out{d_dist, nullptr, d_obj, nullptr, nullptr, nullptr, nullptr, nullptr};
    WHP_CUDA(c, whp_launch_eval(c, d_perms, n_cand, out, (cudaStream_t)cuda_stream));
    return WHP_OK;
  }
  if (c->C > 1024) return fail(c, WHP_ERR_OUT_OF_RANGE, "return / largest-gap routing needs cart_capacity <= 1024");
  WHP_CUDA(c, whp_launch_route(c, d_perms, n_cand, policy, d_dist, d_obj, (cudaStream_t)cuda_stream));
  return WHP_OK;
}

whp_status whp_nhatc_update(whp_ctx* c, const int32_t* d_resp_rows, const int64_t* d_idx,
                            double beta, void* cuda_stream) {
  nvtx_range nvtx_("whp_nhatc_update");
  whp_status s = ready(c);
  if (s != WHP_OK) return s;
  if (!d_resp_rows) return fail(c, WHP_ERR_INVALID_ARG, "d_resp_rows is null");
  if (!std::isfinite(beta) || beta <= 0.0) return fail(c, WHP_ERR_OUT_OF_RANGE, "beta must be finite and positive");
  device_guard dg(c->device);
  WHP_CUDA(c, whp_launch_nhatc_update(c, d_resp_rows, d_idx, beta, (cudaStream_t)cuda_stream));
  return WHP_OK;
}

whp_status whp_nhatc_solve(whp_ctx* c, const int32_t* d_perms, int64_t n_cand, int32_t n_outer,
                           double beta, int64_t* d_idx_hist, int64_t* d_dist_hist,
                           double* d_obj_hist, void* cuda_stream) {
  nvtx_range nvtx_("whp_nhatc_solve");
  whp_status s = ready(c);
  if (s != WHP_OK) return s;
  if (!d_perms || n_cand < 1 || n_outer < 0) return fail(c, WHP_ERR_INVALID_ARG, "bad argument");
  if (!std::isfinite(beta) || beta <= 0.0) return fail(c, WHP_ERR_OUT_OF_RANGE, "beta must be finite and positive");
  device_guard dg(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (c->h_out_cap < n_cand) {
    WHP_CUDA(c, cudaStreamSynchronize(st));
    dfree(c->d_h_dist); dfree(c->d_h_obj);
    WHP_CUDA(c, cudaMalloc(&c->d_h_dist, 8 * (size_t)n_cand));
    WHP_CUDA(c, cudaMalloc(&c->d_h_obj, 8 * (size_t)n_cand));
    c->h_out_cap = n_cand;
  }
  if (c->n_resp_cap < n_cand) {
    WHP_CUDA(c, cudaStreamSynchronize(st));
    dfree(c->d_n_resp);
    WHP_CUDA(c, cudaMalloc(&c->d_n_resp, 4 * (size_t)n_cand * (size_t)c->K));
    c->n_resp_cap = n_cand;
  }
  for (int32_t it = 0; it < n_outer; ++it) {
    if (it == 0) {  // D and r of the plans: once per call, they do not depend on (t, v, w)
      whp_eval_out out{c->d_h_dist, nullptr, c->d_h_obj, nullptr, nullptr, nullptr, nullptr, c->d_n_resp};
      WHP_CUDA(c, whp_launch_eval(c, d_perms, n_cand, out, st));
    } else {        // new multipliers: D6 again on the stored responses
      WHP_CUDA(c, whp_launch_nhatc_rescore(c, c->d_n_resp, c->d_h_dist, n_cand, c->d_h_obj, st));
    }
    WHP_CUDA(c, whp_launch_argmin(c, c->d_h_obj, n_cand, c->d_h_idx, c->d_h_val, st));
    WHP_CUDA(c, whp_launch_nhatc_record(c, c->d_h_idx, c->d_h_dist, c->d_h_obj, it, d_idx_hist,
                                        d_dist_hist, d_obj_hist, st));
    WHP_CUDA(c, whp_launch_nhatc_update(c, c->d_n_resp, c->d_h_idx, beta, st));
  }
  return WHP_OK;
}

whp_status whp_get_penalty(whp_ctx* c, double* t, double* v, double* w, void* cuda_stream) {
  whp_status s = ready(c);
  if (s != WHP_OK) return s;
  device_guard dg(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t bytes = sizeof(double) * (size_t)c->K;
  if (t) WHP_CUDA(c, cudaMemcpyAsync(t, c->d_tvw, bytes, cudaMemcpyDeviceToHost, st));
  if (v) WHP_CUDA(c, cudaMemcpyAsync(v, c->d_tvw + c->K, bytes, cudaMemcpyDeviceToHost, st));
  if (w) WHP_CUDA(c, cudaMemcpyAsync(w, c->d_tvw + 2 * (size_t)c->K, bytes, cudaMemcpyDeviceToHost, st));
  WHP_CUDA(c, cudaStreamSynchronize(st));
  return WHP_OK;
}

whp_status whp_debug_set(whp_ctx* c, int32_t key, int64_t value) {
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  switch (key) {
    case WHP_DEBUG_FORCE_GENERAL: c->dbg_force_general = value > 0 ? 1 : 0; break;
    case WHP_DEBUG_SEGMENTS: c->dbg_segments = value > 0 && value <= 32 ? (int32_t)value : -1; break;
    case WHP_DEBUG_WARPS: c->dbg_warps = value > 0 && value <= 32 ? (int32_t)value : -1; break;
    case WHP_DEBUG_SWAP_MARGIN: c->dbg_swap_margin = value >= 0 ? value : -1; break;
    case WHP_DEBUG_K1_WARPS: c->dbg_k1_warps = value > 0 && value <= 5 ? (int32_t)value : -1; break;
    case WHP_DEBUG_NO_FOURS: c->dbg_no_fours = value > 0 ? 1 : 0; break;
    default: return fail(c, WHP_ERR_INVALID_ARG, "unknown debug key");
  }
  return WHP_OK;
}

whp_status whp_set_swap_stats(whp_ctx* c, int32_t enable) {
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  c->swap_stats = enable != 0;
  return WHP_OK;
}

whp_status whp_get_swap_stats(whp_ctx* c, int64_t* h_batches, int64_t* h_picks, void* cuda_stream) {
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  device_guard dg(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  unsigned long long h[2] = {0, 0};
  WHP_CUDA(c, cudaMemcpyAsync(h, c->d_swap_stats, sizeof(h), cudaMemcpyDeviceToHost, st));
  WHP_CUDA(c, cudaStreamSynchronize(st));
  if (h_batches) *h_batches = (int64_t)h[0];
  if (h_picks) *h_picks = (int64_t)h[1];
  return WHP_OK;
}

whp_status whp_probe_l2_read(whp_ctx* c, int64_t bytes, int32_t reps, float* h_ms) {
  if (!c) return WHP_ERR_INVALID_ARG;
  c->err.clear();
  if (!h_ms || bytes < 16 || reps < 1) return fail(c, WHP_ERR_INVALID_ARG, "bad argument");
  device_guard dg(c->device);
  WHP_CUDA(c, cudaDeviceSynchronize());
  WHP_CUDA(c, whp_launch_l2_probe(c, bytes & ~(int64_t)15, reps, h_ms));
  return WHP_OK;
}

void whp_destroy(whp_ctx* c) {
  if (!c) return;
  {
    device_guard dg(c->device);
    cudaDeviceSynchronize();
    free_orders(c);
    dfree(c->d_tvw); dfree(c->d_argmin_part); dfree(c->d_count); dfree(c->d_task); dfree(c->d_swap_stats);
    dfree(c->d_h_dist); dfree(c->d_h_obj); dfree(c->d_h_idx); dfree(c->d_h_val); dfree(c->d_n_resp);
    for (cudaEvent_t ev : c->ev_piece) cudaEventDestroy(ev);
    for (int k = 0; k < 2; ++k) {
      if (c->s_copy[k]) cudaStreamDestroy(c->s_copy[k]);
      if (c->ev_copied[k]) cudaEventDestroy(c->ev_copied[k]);
      if (c->ev_done[k]) cudaEventDestroy(c->ev_done[k]);
    }
    if (c->s_exec) cudaStreamDestroy(c->s_exec);
  }
  free(c->h_sku_loc); free(c->h_sku_class);
  delete c;
}

}  // extern "C"
