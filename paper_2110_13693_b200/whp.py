"""Thin ctypes binding of libwhp.so (include/whp.h): argument marshalling only — every step of
the path runs in the CUDA kernels. Device arrays are torch tensors (PyTorch is used for device
memory and streams only); host arrays are numpy.

There is no CPU fallback: if libwhp.so has not been built (python -m
paper_2110_13693_b200.build) or cannot be loaded, every call raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libwhp.so")
_lib = None

OK, ERR_INVALID_ARG, ERR_OUT_OF_RANGE, ERR_CAPACITY, ERR_STATE, ERR_CUDA, ERR_NOMEM = range(7)
_STATUS = ["WHP_OK", "WHP_ERR_INVALID_ARG", "WHP_ERR_OUT_OF_RANGE", "WHP_ERR_CAPACITY",
           "WHP_ERR_STATE", "WHP_ERR_CUDA", "WHP_ERR_NOMEM"]

# symbols include/whp.h declares (tests check that the library exports every one)
SYMBOLS = ["whp_create_layout", "whp_load_orders", "whp_set_penalty", "whp_eval_candidates",
           "whp_eval_candidates_host", "whp_eval_swaps", "whp_argmin", "whp_apply_swap",
           "whp_validate_perms", "whp_launch_count", "whp_destroy", "whp_last_error",
           "whp_version", "whp_nhatc_update", "whp_nhatc_solve", "whp_get_penalty",
           "whp_eval_legsum", "whp_kmeans_slotting", "whp_eval_moves", "whp_apply_move",
           "whp_probe_l2_read", "whp_max_batches", "whp_set_swap_stats", "whp_get_swap_stats",
           "whp_debug_set", "whp_eval_routing", "whp_eval_candidates_host16",
           "whp_argmin_static_setup", "whp_argmin_static", "whp_static_last_error"]

ROUTE_S_SHAPE, ROUTE_RETURN, ROUTE_LARGEST_GAP = range(3)
DEBUG_FORCE_GENERAL, DEBUG_SEGMENTS, DEBUG_WARPS, DEBUG_SWAP_MARGIN, DEBUG_K1_WARPS, DEBUG_NO_FOURS = range(6)
ARGMIN_STATIC_MAX_N = 4096 * 4096  # WHP_ARGMIN_STATIC_MAX_N


class WhpError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS[status] if 0 <= status < 7 else status}: {msg}")
        self.status = status


def lib():
    """Load libwhp.so (never builds it, never falls back)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} is missing: run `python -m paper_2110_13693_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(_SO)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.whp_create_layout.argtypes = [i32, i32, i32, i32, i32, i32, vp, vp, i32, i32,
                                        C.POINTER(vp)]
        L.whp_load_orders.argtypes = [vp, i32, vp, vp, i32]
        L.whp_set_penalty.argtypes = [vp, vp, vp, vp]
        L.whp_eval_candidates.argtypes = [vp, vp, i64] + [vp] * 8 + [vp]
        L.whp_eval_candidates_host.argtypes = [vp, vp, i64, vp, vp, vp, vp]
        L.whp_eval_candidates_host16.argtypes = [vp, vp, i64, vp, vp, vp, vp]
        L.whp_eval_swaps.argtypes = [vp, vp, i32, i32, vp, vp, vp]
        L.whp_argmin.argtypes = [vp, vp, i64, vp, vp, vp]
        L.whp_apply_swap.argtypes = [vp, vp, i32, i32, vp, vp]
        L.whp_validate_perms.argtypes = [vp, vp, i64, vp, vp]
        L.whp_nhatc_update.argtypes = [vp, vp, vp, C.c_double, vp]
        L.whp_nhatc_solve.argtypes = [vp, vp, i64, i32, C.c_double, vp, vp, vp, vp]
        L.whp_get_penalty.argtypes = [vp, vp, vp, vp, vp]
        L.whp_eval_legsum.argtypes = [vp, vp, i64, vp, vp]
        L.whp_eval_routing.argtypes = [vp, vp, i64, i32, vp, vp, vp]
        L.whp_kmeans_slotting.argtypes = [i32, i32, i32, i32, vp, i32, i32, i32, i32, i32, vp, vp, vp, vp]
        L.whp_eval_moves.argtypes = [vp, vp, i32, i32, vp, vp, vp]
        L.whp_apply_move.argtypes = [vp, vp, i32, i32, vp, vp]
        L.whp_probe_l2_read.argtypes = [vp, i64, i32, vp]
        L.whp_set_swap_stats.argtypes = [vp, i32]
        L.whp_debug_set.argtypes = [vp, i32, i64]
        L.whp_get_swap_stats.argtypes = [vp, vp, vp, vp]
        L.whp_max_batches.argtypes = [vp]
        L.whp_max_batches.restype = i64
        L.whp_launch_count.argtypes = [vp]
        L.whp_launch_count.restype = i64
        L.whp_destroy.argtypes = [vp]
        L.whp_destroy.restype = None
        L.whp_last_error.argtypes = [vp]
        L.whp_last_error.restype = C.c_char_p
        L.whp_version.restype = C.c_char_p
        L.whp_argmin_static_setup.argtypes = []
        L.whp_argmin_static.argtypes = [vp, i64, vp, vp, vp]
        L.whp_static_last_error.argtypes = []
        L.whp_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _h(a, dtype):
    """host numpy array -> (keepalive, pointer)"""
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data


def _d(t, dtype=None, numel=None, device=None):
    """device torch tensor -> raw pointer (None -> NULL). Checks what the C side cannot see:
    contiguity, dtype, at least `numel` elements, and the context's device."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
    if numel is not None and t.numel() < numel:
        raise ValueError(f"tensor has {t.numel()} elements, the call writes / reads {numel}")
    if device is not None and t.device.index != device:
        raise ValueError(f"tensor lives on cuda:{t.device.index}, the context on cuda:{device}")
    return t.data_ptr()


def _hostbuf(a, np_dtype, numel, name):
    """host numpy array or CPU torch tensor -> raw pointer, after checking dtype / size /
    contiguity (a mismatch would be silently misread by the C side)."""
    if a is None:
        return None
    if hasattr(a, "data_ptr"):  # torch CPU tensor
        import torch
        want = {np.int32: torch.int32, np.int64: torch.int64, np.float64: torch.float64}[np_dtype]
        if a.is_cuda or not a.is_contiguous() or a.dtype != want or a.numel() < numel:
            raise ValueError(f"{name}: expected a contiguous CPU tensor of {want} with >= {numel} elements")
        return a.data_ptr()
    if not isinstance(a, np.ndarray) or a.dtype != np_dtype or not a.flags.c_contiguous or a.size < numel:
        raise ValueError(f"{name}: expected a C-contiguous numpy array of {np.dtype(np_dtype)} "
                         f"with >= {numel} elements")
    return a.ctypes.data


def _stream(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream


class Context:
    """Owns one whp_ctx. Method names are the C entry points without the `whp_` prefix."""

    def __init__(self, n_aisles, slots_per_side, slot_pitch, aisle_spacing, depot_aisle,
                 sku_loc, sku_class, n_classes, device=0):
        L = lib()
        k1, p_loc = _h(sku_loc, np.int32)
        k2, p_cls = _h(sku_class, np.int32)
        if k1 is None or k2 is None or len(k1) != len(k2):
            raise WhpError(ERR_INVALID_ARG, "sku_loc / sku_class")
        h = C.c_void_p()
        st = L.whp_create_layout(n_aisles, slots_per_side, slot_pitch, aisle_spacing,
                                 depot_aisle, len(k1), p_loc, p_cls, n_classes, device,
                                 C.byref(h))
        if st != OK:
            raise WhpError(st, "whp_create_layout")
        self._h = h
        self.device = device
        self.n_classes = n_classes
        self.n_orders = 0

    @classmethod
    def from_problem(cls, pb, device=0):
        """pb: workloads.Problem (or anything with its attributes)."""
        ctx = cls(pb.n_aisles, pb.slots_per_side, pb.slot_pitch, pb.aisle_spacing,
                  pb.depot_aisle, pb.sku_loc, pb.sku_class, pb.n_classes, device)
        ctx.load_orders(pb.order_ptr, pb.item_sku, pb.cart_capacity)
        ctx.set_penalty(pb.t, pb.v, pb.w)
        return ctx

    def _check(self, st):
        if st != OK:
            raise WhpError(st, lib().whp_last_error(self._h).decode())

    def load_orders(self, order_ptr, item_sku, cart_capacity):
        k1, p1 = _h(order_ptr, np.int32)
        k2, p2 = _h(item_sku, np.int32)
        n_orders = len(k1) - 1
        if n_orders >= 1 and len(k2) != int(k1[-1]):
            raise WhpError(ERR_INVALID_ARG, "len(item_sku) != order_ptr[-1]")
        self._check(lib().whp_load_orders(self._h, n_orders, p1, p2, cart_capacity))
        self.n_orders = n_orders

    def set_penalty(self, t, v, w):
        ks = [_h(x, np.float64) for x in (t, v, w)]
        if any(k[0] is None or len(k[0]) != self.n_classes for k in ks):
            raise WhpError(ERR_INVALID_ARG, "t, v, w must have n_classes entries")
        self._check(lib().whp_set_penalty(self._h, ks[0][1], ks[1][1], ks[2][1]))

    def eval_candidates(self, perms, dist=None, penalty=None, obj=None, n_batches=None,
                        batch_hash=None, batch_of_pos=None, n_distinct=None, resp=None,
                        stream=None):
        """perms: CUDA int32 [n_cand][n_orders]; outputs are caller-allocated CUDA tensors."""
        import torch
        n_cand = perms.shape[0] if perms.dim() == 2 else 1
        if perms.numel() != n_cand * self.n_orders:
            raise WhpError(ERR_INVALID_ARG, "perms shape")
        dv, K, n = self.device, self.n_classes, self.n_orders
        self._check(lib().whp_eval_candidates(
            self._h, _d(perms, torch.int32, n_cand * n, dv), n_cand,
            _d(dist, torch.int64, n_cand, dv), _d(penalty, torch.float64, n_cand, dv),
            _d(obj, torch.float64, n_cand, dv), _d(n_batches, torch.int32, n_cand, dv),
            _d(batch_hash, torch.int64, n_cand, dv), _d(batch_of_pos, torch.int32, n_cand * n, dv),
            _d(n_distinct, torch.int32, n_cand, dv), _d(resp, torch.int32, n_cand * K, dv),
            _stream(stream)))

    def eval_candidates_host(self, perms, dist=None, obj=None, want_argmin=True):
        """perms / dist / obj: host numpy arrays or CPU torch tensors (pinned = async copies).
        int32 plans go through whp_eval_candidates_host, uint16 plans (numpy uint16, torch
        uint16 / int16 bit patterns) through whp_eval_candidates_host16.
        Returns (argmin_idx, argmin_val) when want_argmin."""
        n_cand = perms.shape[0]
        if tuple(perms.shape) != (n_cand, self.n_orders):
            raise WhpError(ERR_INVALID_ARG, "perms shape")
        is16 = (perms.dtype == np.uint16) if isinstance(perms, np.ndarray) else \
            (str(perms.dtype) in ("torch.uint16", "torch.int16"))
        fn = lib().whp_eval_candidates_host16 if is16 else lib().whp_eval_candidates_host
        if is16 and not isinstance(perms, np.ndarray):
            if perms.is_cuda or not perms.is_contiguous():
                raise ValueError("perms: expected a contiguous CPU tensor")
            p_perms = perms.data_ptr()
        else:
            p_perms = _hostbuf(perms, np.uint16 if is16 else np.int32, n_cand * self.n_orders, "perms")
        p_dist = _hostbuf(dist, np.int64, n_cand, "dist")
        p_obj = _hostbuf(obj, np.float64, n_cand, "obj")
        idx, val = C.c_int64(-1), C.c_double(0.0)
        self._check(fn(
            self._h, p_perms, n_cand, p_dist, p_obj,
            C.addressof(idx) if want_argmin else None,
            C.addressof(val) if want_argmin else None))
        return (idx.value, val.value) if want_argmin else None

    def eval_swaps(self, base_perm, win_start, win_len, dist=None, obj=None, stream=None):
        import torch
        nn, dv = win_len * (win_len - 1) // 2, self.device
        self._check(lib().whp_eval_swaps(self._h, _d(base_perm, torch.int32, self.n_orders, dv),
                                         win_start, win_len, _d(dist, torch.int64, nn, dv),
                                         _d(obj, torch.float64, nn, dv), _stream(stream)))

    def argmin(self, obj, idx, val=None, n=None, stream=None):
        import torch
        n = obj.numel() if n is None else n
        dv = self.device
        self._check(lib().whp_argmin(self._h, _d(obj, torch.float64, n, dv), n,
                                     _d(idx, torch.int64, 1, dv), _d(val, torch.float64, 1, dv),
                                     _stream(stream)))

    def apply_swap(self, base_perm, win_start, win_len, idx, stream=None):
        import torch
        dv = self.device
        self._check(lib().whp_apply_swap(self._h, _d(base_perm, torch.int32, self.n_orders, dv),
                                         win_start, win_len, _d(idx, torch.int64, 1, dv),
                                         _stream(stream)))

    def eval_moves(self, base_perm, win_start, win_len, dist=None, obj=None, stream=None):
        """NEXT-4 (reading N4): all W(W-1) insertion moves inside the window."""
        import torch
        nn, dv = win_len * (win_len - 1), self.device
        self._check(lib().whp_eval_moves(self._h, _d(base_perm, torch.int32, self.n_orders, dv),
                                         win_start, win_len, _d(dist, torch.int64, nn, dv),
                                         _d(obj, torch.float64, nn, dv), _stream(stream)))

    def apply_move(self, base_perm, win_start, win_len, idx, stream=None):
        import torch
        dv = self.device
        self._check(lib().whp_apply_move(self._h, _d(base_perm, torch.int32, self.n_orders, dv),
                                         win_start, win_len, _d(idx, torch.int64, 1, dv),
                                         _stream(stream)))

    def eval_legsum(self, perms, length, stream=None):
        """NEXT-2 (reading N2): summed leg lengths of every plan into `length` (CUDA int64)."""
        import torch
        n_cand = perms.shape[0] if perms.dim() == 2 else 1
        dv = self.device
        self._check(lib().whp_eval_legsum(self._h, _d(perms, torch.int32, n_cand * self.n_orders, dv),
                                          n_cand, _d(length, torch.int64, n_cand, dv),
                                          _stream(stream)))

    def eval_routing(self, perms, policy, dist=None, obj=None, stream=None):
        """NEXT-2 (readings N5 / N6): D and J of every plan with its carts routed by `policy`
        (ROUTE_S_SHAPE, ROUTE_RETURN, ROUTE_LARGEST_GAP)."""
        import torch
        n_cand = perms.shape[0] if perms.dim() == 2 else 1
        dv = self.device
        self._check(lib().whp_eval_routing(self._h, _d(perms, torch.int32, n_cand * self.n_orders, dv),
                                           n_cand, int(policy), _d(dist, torch.int64, n_cand, dv),
                                           _d(obj, torch.float64, n_cand, dv), _stream(stream)))

    def nhatc_update(self, resp_rows, idx=None, beta=1.0, stream=None):
        """NEXT-1 (reading N1): v <- v + 2 w^2 (t - r*), w <- beta w; r* = row idx[0] of resp_rows."""
        import torch
        dv = self.device
        self._check(lib().whp_nhatc_update(self._h, _d(resp_rows, torch.int32, self.n_classes, dv),
                                           _d(idx, torch.int64, 1, dv), float(beta), _stream(stream)))

    def nhatc_solve(self, perms, n_outer, beta, idx_hist=None, dist_hist=None, obj_hist=None,
                    stream=None):
        """n_outer x {eval_candidates -> argmin -> record -> nhatc_update}, all on the device."""
        import torch
        n_cand = perms.shape[0]
        dv, no = self.device, int(n_outer)
        self._check(lib().whp_nhatc_solve(self._h, _d(perms, torch.int32, n_cand * self.n_orders, dv),
                                          n_cand, no, float(beta), _d(idx_hist, torch.int64, no, dv),
                                          _d(dist_hist, torch.int64, no, dv),
                                          _d(obj_hist, torch.float64, no, dv), _stream(stream)))

    def get_penalty(self, stream=None):
        t, v, w = (np.zeros(self.n_classes, np.float64) for _ in range(3))
        self._check(lib().whp_get_penalty(self._h, t.ctypes.data, v.ctypes.data, w.ctypes.data,
                                          _stream(stream)))
        return t, v, w

    def validate_perms(self, perms, stream=None) -> int:
        import torch
        n_bad = C.c_int64(0)
        self._check(lib().whp_validate_perms(self._h, _d(perms, torch.int32, perms.shape[0] * self.n_orders,
                                                         self.device), perms.shape[0],
                                             C.addressof(n_bad), _stream(stream)))
        return n_bad.value

    def probe_l2_read(self, nbytes=32 << 20, reps=200) -> float:
        """Measured L2 read bandwidth in GB/s (read-only sweeps of an L2-resident buffer)."""
        ms = C.c_float(0.0)
        self._check(lib().whp_probe_l2_read(self._h, nbytes, reps, C.byref(ms)))
        return nbytes * reps / (ms.value * 1e-3) / 1e9

    def set_swap_stats(self, enable=True):
        self._check(lib().whp_set_swap_stats(self._h, 1 if enable else 0))

    def get_swap_stats(self, stream=None):
        """(batches, picks) scored from their picks by the latest eval_swaps / eval_moves call
        made while the statistics were enabled."""
        b, k = C.c_int64(0), C.c_int64(0)
        self._check(lib().whp_get_swap_stats(self._h, C.addressof(b), C.addressof(k),
                                             _stream(stream)))
        return b.value, k.value

    def debug_set(self, key: int, value: int = -1):
        """Kernel-selection switch for tests / measurements (whp.h: whp_debug_set); value < 0 =
        default."""
        self._check(lib().whp_debug_set(self._h, int(key), int(value)))

    def max_batches(self) -> int:
        return int(lib().whp_max_batches(self._h))

    def launch_count(self) -> int:
        return int(lib().whp_launch_count(self._h))

    def close(self):
        if getattr(self, "_h", None):
            lib().whp_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def kmeans_slotting(n_aisles, slots_per_side, depot_aisle, n_skus, item_sku, k, n_zones, iters,
                    device=0) -> dict:
    """NEXT-3 (reading N3): K-means of the SKUs on their pick frequency + cluster-contiguous
    slotting, on the GPU. Returns sku_loc, sku_class (inputs of Context(...)), assign, centroids."""
    k1, p1 = _h(item_sku, np.int32)
    out = {"sku_loc": np.zeros(n_skus, np.int32), "sku_class": np.zeros(n_skus, np.int32),
           "assign": np.zeros(n_skus, np.int32), "centroids": np.zeros(k, np.float64)}
    st = lib().whp_kmeans_slotting(n_aisles, slots_per_side, depot_aisle, n_skus, p1, len(k1), k,
                                   n_zones, iters, device, out["sku_loc"].ctypes.data,
                                   out["sku_class"].ctypes.data, out["assign"].ctypes.data,
                                   out["centroids"].ctypes.data)
    if st != OK:
        raise WhpError(st, "whp_kmeans_slotting")
    return out


def _check_static(st):
    if st != OK:
        raise WhpError(st, lib().whp_static_last_error().decode())


def argmin_static_setup():
    """whp_argmin_static_setup: resolve the static scratch's address on torch's current device
    (once per device; needed beforehand only when the first whp_argmin_static would be captured)."""
    _check_static(lib().whp_argmin_static_setup())


def argmin_static(obj, idx, val=None, n=None, stream=None):
    """whp_argmin_static: D7 without a context and without any allocation, n <=
    ARGMIN_STATIC_MAX_N; the tensors must live on torch's current device. Calls that overlap on
    the GPU race on the shared static scratch."""
    import torch
    n = obj.numel() if n is None else n
    dv = torch.cuda.current_device()
    _check_static(lib().whp_argmin_static(_d(obj, torch.float64, n, dv), n,
                                          _d(idx, torch.int64, 1, dv),
                                          _d(val, torch.float64, 1, dv), _stream(stream)))


def version() -> str:
    return lib().whp_version().decode()
