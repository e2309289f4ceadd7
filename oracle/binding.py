"""ctypes marshalling for whp_oracle.c. The arithmetic of the method lives in the C file; the only
compositions written here are `nhatc_loop` (the outer loop of reading N1: eval -> argmin -> update,
each step a C routine) and the `threads=` wrappers, which spread candidates / neighbourhood rows
over host threads around the same single-threaded C routines ("wrapper only")."""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "whp_oracle.c")
_SO = os.path.join(_HERE, "libwhp_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off: every fp64 * and + individually rounded (reading Q12)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-shared",
             "-fPIC", "-o", _SO, _SRC])
    return _SO


class _Geom(C.Structure):
    _fields_ = [("n_aisles", C.c_int32), ("slots_per_side", C.c_int32),
                ("slot_pitch", C.c_int32), ("aisle_spacing", C.c_int32),
                ("depot_aisle", C.c_int32)]


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_batch_distance.restype = C.c_int64
        _lib.orc_optimal_route.restype = C.c_int64
        _lib.orc_penalty.restype = C.c_double
        _lib.orc_argmin.restype = C.c_int64
        _lib.orc_tour_length.restype = C.c_int64
        _lib.orc_batch_return_distance.restype = C.c_int64
        _lib.orc_batch_largest_gap_distance.restype = C.c_int64
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _geom(g):
    """g: any object with the five geometry attributes (e.g. workloads.Problem), or a 5-tuple
    (n_aisles, slots_per_side, slot_pitch, aisle_spacing, depot_aisle)."""
    if hasattr(g, "n_aisles"):
        return _Geom(int(g.n_aisles), int(g.slots_per_side), int(g.slot_pitch),
                     int(g.aisle_spacing), int(g.depot_aisle))
    return _Geom(*[int(x) for x in g])


def batch_distance(geom, locs) -> int:
    locs = _i32(locs)
    return int(_load().orc_batch_distance(C.byref(_geom(geom)), _p(locs), C.c_int32(len(locs))))


def optimal_route(geom, locs) -> int:
    locs = _i32(locs)
    return int(_load().orc_optimal_route(C.byref(_geom(geom)), _p(locs), C.c_int32(len(locs))))


def penalty(r, t, v, w) -> float:
    r, t, v, w = _i32(r), _f64(t), _f64(v), _f64(w)
    return float(_load().orc_penalty(C.c_int32(len(r)), _p(r), _p(t), _p(v), _p(w)))


def argmin(x) -> int:
    x = _f64(x)
    return int(_load().orc_argmin(_p(x), C.c_int64(len(x))))


def decode_neighbour(W: int, n: int):
    i, j = C.c_int32(), C.c_int32()
    _load().orc_decode_neighbour(C.c_int32(W), C.c_int64(n), C.byref(i), C.byref(j))
    return i.value, j.value


def _common(pb):
    keep = (_i32(pb.sku_loc), _i32(pb.sku_class), _i32(pb.order_ptr), _i32(pb.item_sku),
            _f64(pb.t), _f64(pb.v), _f64(pb.w))
    g = _geom(pb)
    args = [C.byref(g), _p(keep[0]), _p(keep[1]), C.c_int32(pb.n_classes),
            C.c_int32(pb.n_orders), _p(keep[2]), _p(keep[3]), C.c_int32(pb.cart_capacity),
            _p(keep[4]), _p(keep[5]), _p(keep[6])]
    return args, (keep, g)


def _pool_map(fn, cuts, threads):
    """fn(lo, hi) over consecutive cuts on `threads` host threads (the C routines release the GIL)."""
    from concurrent.futures import ThreadPoolExecutor
    spans = [(int(cuts[k]), int(cuts[k + 1])) for k in range(len(cuts) - 1) if cuts[k] < cuts[k + 1]]
    with ThreadPoolExecutor(max(1, threads)) as ex:
        list(ex.map(lambda ab: fn(*ab), spans))


def _off(a, row):
    """pointer to row `row` of a C-contiguous array (None stays NULL)"""
    return None if a is None else C.c_void_p(a.ctypes.data + int(row) * a.strides[0])


def eval_candidates(pb, perms, detail: bool = False, threads: int = 1) -> dict:
    """D1–D6 for every row of perms. detail=True also returns batch_of_pos and resp.
    threads > 1: candidate slices on that many host threads, same routine per candidate."""
    perms = _i32(perms)
    if perms.ndim == 1:
        perms = perms[None, :]
    n_cand, n = perms.shape
    assert n == pb.n_orders
    out = {
        "dist": np.zeros(n_cand, np.int64), "penalty": np.zeros(n_cand, np.float64),
        "obj": np.zeros(n_cand, np.float64), "n_batches": np.zeros(n_cand, np.int32),
        "batch_hash": np.zeros(n_cand, np.uint64), "n_distinct": np.zeros(n_cand, np.int32),
        "batch_of_pos": np.zeros((n_cand, n), np.int32) if detail else None,
        "resp": np.zeros((n_cand, pb.n_classes), np.int32) if detail else None,
    }
    args, keep = _common(pb)
    lib = _load()

    def run(lo, hi):
        lib.orc_eval_candidates(*args, _off(perms, lo), C.c_int64(hi - lo), _off(out["dist"], lo),
                                _off(out["penalty"], lo), _off(out["obj"], lo),
                                _off(out["n_batches"], lo), _off(out["batch_hash"], lo),
                                _off(out["batch_of_pos"], lo), _off(out["n_distinct"], lo),
                                _off(out["resp"], lo))
    if threads <= 1:
        run(0, n_cand)
    else:
        _pool_map(run, np.linspace(0, n_cand, min(n_cand, 8 * threads) + 1).astype(np.int64), threads)
    del keep
    return out


def eval_candidate_batches(pb, perm):
    """Per-batch S-shape lengths of one plan (for the brute-force bound P3)."""
    perm = _i32(perm)
    nb = C.c_int32()
    bd = np.zeros(pb.n_orders, np.int64)
    bop = np.zeros(pb.n_orders, np.int32)
    args, keep = _common(pb)
    _load().orc_eval_candidate(*args, _p(perm), None, None, None, C.byref(nb), None, _p(bop),
                               None, None, _p(bd))
    del keep
    return bd[:nb.value].copy(), bop


def eval_swaps(pb, base_perm, win_start: int, win_len: int, threads: int = 1) -> dict:
    """D8: every pairwise swap inside the window, each materialised and evaluated from scratch.
    threads > 1: the rows i' of the neighbourhood on that many host threads."""
    base_perm = _i32(base_perm)
    nn = win_len * (win_len - 1) // 2
    out = {"dist": np.zeros(nn, np.int64), "obj": np.zeros(nn, np.float64)}
    args, keep = _common(pb)
    lib = _load()
    if threads <= 1:
        lib.orc_eval_swaps(*args, _p(base_perm), C.c_int32(win_start), C.c_int32(win_len),
                           _p(out["dist"]), _p(out["obj"]))
    else:
        def run(lo, hi):
            lib.orc_eval_swaps_rows(*args, _p(base_perm), C.c_int32(win_start),
                                    C.c_int32(win_len), C.c_int32(lo), C.c_int32(hi),
                                    _p(out["dist"]), _p(out["obj"]))
        # row i' holds W-1-i' neighbours: pair row k with row W-2-k so every task is equal
        half = (win_len - 1 + 1) // 2
        from concurrent.futures import ThreadPoolExecutor
        def pair(k):
            run(k, k + 1)
            m = win_len - 2 - k
            if m > k:
                run(m, m + 1)
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(pair, range(half)))
    del keep
    return out


def swap_trajectory(pb, base_perm, W: int, stride: int, n_iter: int) -> dict:
    perm = _i32(base_perm).copy()
    out = {"move": np.zeros(n_iter, np.int64), "dist": np.zeros(n_iter, np.int64),
           "obj": np.zeros(n_iter, np.float64)}
    args, keep = _common(pb)
    _load().orc_swap_trajectory(*args, _p(perm), C.c_int32(W), C.c_int32(stride),
                                C.c_int32(n_iter), _p(out["move"]), _p(out["dist"]),
                                _p(out["obj"]))
    del keep
    out["perm"] = perm
    return out


def nhatc_update(r, t, v, w, beta: float):
    """Reading N1: v <- v + 2 w^2 (t - r), w <- beta w. Returns new (v, w)."""
    r, t = _i32(r), _f64(t)
    v, w = _f64(v).copy(), _f64(w).copy()
    _load().orc_nhatc_update(C.c_int32(len(r)), _p(r), _p(t), _p(v), _p(w), C.c_double(beta))
    return v, w


def nhatc_loop(pb, perms, n_outer: int, beta: float) -> dict:
    """NEXT-1: n_outer times {score every plan (D1-D6), take the argmin (D7), read its
    responses r*, update the multipliers (N1)}. Returns the per-iteration winner, its D and J,
    and the final v, w."""
    import copy
    pb = copy.copy(pb)
    pb.v, pb.w = _f64(pb.v).copy(), _f64(pb.w).copy()
    hist = {"idx": np.zeros(n_outer, np.int64), "dist": np.zeros(n_outer, np.int64),
            "obj": np.zeros(n_outer, np.float64)}
    for it in range(n_outer):
        out = eval_candidates(pb, perms)
        i = argmin(out["obj"])
        one = eval_candidates(pb, _i32(perms)[i], detail=True)
        hist["idx"][it], hist["dist"][it], hist["obj"][it] = i, out["dist"][i], out["obj"][i]
        pb.v, pb.w = nhatc_update(one["resp"][0], pb.t, pb.v, pb.w, beta)
    hist["v"], hist["w"] = pb.v, pb.w
    return hist


def tour_length(geom, locs) -> int:
    """NEXT-2: depot -> locs in the given order -> depot under D0's walking metric."""
    locs = _i32(locs)
    return int(_load().orc_tour_length(C.byref(_geom(geom)), _p(locs), C.c_int32(len(locs))))


def eval_legsum(pb, perms) -> np.ndarray:
    """NEXT-2 (reading N2): summed leg lengths of every plan, carts by next-fit (D2)."""
    perms = _i32(perms)
    if perms.ndim == 1:
        perms = perms[None, :]
    n_cand = perms.shape[0]
    out = np.zeros(n_cand, np.int64)
    g = _geom(pb)
    keep = (_i32(pb.sku_loc), _i32(pb.order_ptr), _i32(pb.item_sku))
    _load().orc_eval_legsum(C.byref(g), _p(keep[0]), C.c_int32(pb.n_orders), _p(keep[1]),
                            _p(keep[2]), C.c_int32(pb.cart_capacity), _p(perms),
                            C.c_int64(n_cand), _p(out))
    return out


def kmeans_slotting(geom, n_skus: int, item_sku, k: int, Z: int, iters: int) -> dict:
    """NEXT-3 (reading N3): K-means of the SKUs on their pick frequency, then cluster-contiguous
    slotting. Returns sku_loc, sku_class, assign, centroids, freq."""
    item_sku = _i32(item_sku)
    out = {"sku_loc": np.zeros(n_skus, np.int32), "sku_class": np.zeros(n_skus, np.int32),
           "assign": np.zeros(n_skus, np.int32), "centroids": np.zeros(k, np.float64),
           "freq": np.zeros(n_skus, np.int64)}
    g = _geom(geom)
    st = _load().orc_kmeans_slotting(C.byref(g), C.c_int32(n_skus), _p(item_sku),
                                     C.c_int32(len(item_sku)), C.c_int32(k), C.c_int32(Z),
                                     C.c_int32(iters), _p(out["sku_loc"]), _p(out["sku_class"]),
                                     _p(out["assign"]), _p(out["centroids"]), _p(out["freq"]))
    if st != 0:
        raise ValueError("kmeans_slotting: bad arguments")
    return out


def eval_moves(pb, base_perm, win_start: int, win_len: int) -> dict:
    """NEXT-4 (reading N4): every insertion move (i' -> j') inside the window, W(W-1) of them."""
    base_perm = _i32(base_perm)
    nn = win_len * (win_len - 1)
    out = {"dist": np.zeros(nn, np.int64), "obj": np.zeros(nn, np.float64)}
    args, keep = _common(pb)
    _load().orc_eval_moves(*args, _p(base_perm), C.c_int32(win_start), C.c_int32(win_len),
                           _p(out["dist"]), _p(out["obj"]))
    del keep
    return out


S_SHAPE, RETURN, LARGEST_GAP = 0, 1, 2  # routing policies (D4, readings N5 and N6)


def batch_return_distance(geom, locs) -> int:
    """NEXT-2 (reading N5): return routing of one cart."""
    locs = _i32(locs)
    return int(_load().orc_batch_return_distance(C.byref(_geom(geom)), _p(locs), C.c_int32(len(locs))))


def batch_largest_gap_distance(geom, locs) -> int:
    """NEXT-2 (reading N6): largest-gap routing of one cart."""
    locs = _i32(locs)
    return int(_load().orc_batch_largest_gap_distance(C.byref(_geom(geom)), _p(locs),
                                                      C.c_int32(len(locs))))


def eval_routing(pb, perms, policy: int, threads: int = 1) -> dict:
    """D and J = D + phi of every plan with the carts routed by `policy` (0 S-shape, 1 return,
    2 largest gap); batching, responses and penalty as in eval_candidates."""
    perms = _i32(perms)
    if perms.ndim == 1:
        perms = perms[None, :]
    n_cand = perms.shape[0]
    out = {"dist": np.zeros(n_cand, np.int64), "obj": np.zeros(n_cand, np.float64)}
    args, keep = _common(pb)
    lib = _load()

    def run(lo, hi):
        st = lib.orc_eval_routing(*args, C.c_int32(policy), _off(perms, lo), C.c_int64(hi - lo),
                                  _off(out["dist"], lo), _off(out["obj"], lo))
        if st != 0:
            raise ValueError("eval_routing: unknown policy")
    if threads <= 1:
        run(0, n_cand)
    else:
        _pool_map(run, np.linspace(0, n_cand, min(n_cand, 8 * threads) + 1).astype(np.int64), threads)
    del keep
    return out
