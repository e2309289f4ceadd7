"""Seeded synthetic workloads — the ONLY module shared by the CUDA path's tests/bench and the
oracle. It holds no arithmetic of the method (no batching, routing, penalty or argmin): it
only draws inputs shaped like the paper's workload statement (§1: ~10,000 items,
4,000 orders, 200,000 locations per day) in the five configurations BASELINE.json lists.
The company's real order data is private; these are stand-ins (DESIGN.md §4 has the recipe).

Everything is a pure function of (config name, seed): integer streams come from splitmix64
counters, one sub-stream per array, so any slice (e.g. one candidate permutation out of
65,536) can be regenerated on the CPU with numpy or on the GPU with torch, bit-identically.
"""
from dataclasses import dataclass, field

import numpy as np

_M64 = (1 << 64) - 1
_GAMMA = 0x9E3779B97F4A7C15
_MUL1 = 0xBF58476D1CE4E5B9
_MUL2 = 0x94D049BB133111EB


def splitmix64(x):
    """One splitmix64 output step on a uint64 array (Steele, Lea & Flood 2014)."""
    with np.errstate(over="ignore"):
        z = np.asarray(x, dtype=np.uint64) + np.uint64(_GAMMA)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(_MUL1)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(_MUL2)
        return z ^ (z >> np.uint64(31))


def _sub_seed(seed: int, sub: int) -> np.uint64:
    return splitmix64(np.uint64(((seed * 0x100000001B3) ^ (sub * 0x9E3779B1)) & _M64))


def stream_u64(seed: int, sub: int, n: int, start: int = 0):
    """u64 stream: element i = splitmix64(sub_seed + i)."""
    with np.errstate(over="ignore"):
        return splitmix64(_sub_seed(seed, sub) + np.arange(start, start + n, dtype=np.uint64))


def stream_u01(seed: int, sub: int, n: int):
    """fp64 uniforms in [0,1) with 53 random bits."""
    return (stream_u64(seed, sub, n) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def _shuffle(seed: int, sub: int, n: int):
    """Seeded random permutation of 0..n-1 (stable argsort of random keys)."""
    return np.argsort(stream_u64(seed, sub, n), kind="stable").astype(np.int64)


# sub-stream ids
_S_PLACE, _S_RANK, _S_COUNT, _S_SKU, _S_T, _S_V, _S_W, _S_PERM, _S_BASE = range(1, 10)


@dataclass
class Problem:
    """Exactly the arrays whp_create_layout / whp_load_orders / whp_set_penalty take."""
    n_aisles: int
    slots_per_side: int
    slot_pitch: int
    aisle_spacing: int
    depot_aisle: int
    sku_loc: np.ndarray
    sku_class: np.ndarray
    n_classes: int
    order_ptr: np.ndarray
    item_sku: np.ndarray
    cart_capacity: int
    t: np.ndarray
    v: np.ndarray
    w: np.ndarray

    @property
    def n_orders(self) -> int:
        return len(self.order_ptr) - 1

    @property
    def n_items(self) -> int:
        return int(self.order_ptr[-1])

    @property
    def n_skus(self) -> int:
        return len(self.sku_loc)


@dataclass
class Workload:
    name: str
    problem: Problem
    n_cand: int
    seed: int = 0
    # config 4 (swap neighbourhood trajectory)
    window: int = 0
    stride: int = 0
    n_iter: int = 0
    meta: dict = field(default_factory=dict)


CONFIGS = {
    # name: geometry, SKUs, categories x zones, orders, item-count law, capacity, candidates
    "tiny": dict(NA=4, S=10, n_skus=40, n_cat=4, Z=1, K=4, n_orders=20, count=("uniform", 1, 4),
                 zipf=None, C=8, n_cand=64, clustered=False, t_hi="ten", vw="unit"),
    "mid": dict(NA=20, S=50, n_skus=2000, n_cat=10, Z=2, K=20, n_orders=500,
                count=("geom", 0.4, 10), zipf=1.0, C=20, n_cand=4096, clustered=True,
                t_hi="batches", vw="unit"),
    "paper": dict(NA=400, S=250, n_skus=100000, n_cat=50, Z=4, K=200, n_orders=4000,
                  count=("geom", 0.4, 30), zipf=1.0, C=30, n_cand=16384, clustered=True,
                  t_hi="batches", vw="unit"),
    "stress": dict(NA=400, S=250, n_skus=100000, n_cat=50, Z=4, K=32, n_orders=20000,
                   count=("geom", 0.3, 20), zipf=1.2, C=40, n_cand=65536, clustered=True,
                   t_hi="batches", vw="log"),
}
CONFIGS["neighbourhood"] = dict(CONFIGS["paper"], n_cand=1, window=256, stride=128, n_iter=100)


def make_problem(name: str, seed: int = 0, **override) -> Problem:
    """Draw the layout, SKU tables, orders and penalty parameters of a named config."""
    cfg = dict(CONFIGS[name], **override)
    NA, S, n_skus, n_cat, Z, K = (cfg[k] for k in ("NA", "S", "n_skus", "n_cat", "Z", "K"))
    per_cat = n_skus // n_cat
    category = np.arange(n_skus, dtype=np.int64) // per_cat  # reading Q19
    sku_loc = np.empty(n_skus, dtype=np.int64)
    if cfg["clustered"]:
        # category g owns a contiguous block of aisles; distinct random slots inside it
        aisles_per_cat = NA // n_cat
        block = aisles_per_cat * 2 * S
        assert per_cat <= block
        for g in range(n_cat):
            order = _shuffle(seed, _S_PLACE * 1000 + g, block)[:per_cat]
            sku_loc[g * per_cat:(g + 1) * per_cat] = g * block + order
    else:
        sku_loc[:] = _shuffle(seed, _S_PLACE, 2 * NA * S)[:n_skus]
    slot = sku_loc % S
    zone = slot * Z // S  # depth bands (reading Q10)
    if K == n_cat * Z:
        sku_class = category * Z + zone
    else:  # stress: 32 classes = (category mod 8) x 4 zones
        sku_class = (category % (K // Z)) * Z + zone

    # order sizes
    n_orders = cfg["n_orders"]
    law = cfg["count"]
    u = stream_u01(seed, _S_COUNT, n_orders)
    if law[0] == "uniform":
        q = law[1] + np.floor(u * (law[2] - law[1] + 1)).astype(np.int64)
    else:  # 1 + Geometric(p) on {0,1,...}, capped (reading Q17)
        p = law[1]
        q = 1 + np.floor(np.log1p(-u) / np.log1p(-p)).astype(np.int64)
        q = np.minimum(q, min(law[2], cfg["C"]))
    order_ptr = np.zeros(n_orders + 1, dtype=np.int64)
    np.cumsum(q, out=order_ptr[1:])
    n_items = int(order_ptr[-1])

    # SKU of every item: uniform, or Zipf(s) over a seeded random ranking (reading Q18)
    ui = stream_u01(seed, _S_SKU, n_items)
    if cfg["zipf"] is None:
        item_sku = np.floor(ui * n_skus).astype(np.int64)
    else:
        wts = 1.0 / np.arange(1, n_skus + 1, dtype=np.float64) ** cfg["zipf"]
        cdf = np.cumsum(wts)
        rank = np.searchsorted(cdf, ui * cdf[-1], side="right")
        rank = np.minimum(rank, n_skus - 1)
        sku_of_rank = _shuffle(seed, _S_RANK, n_skus)
        item_sku = sku_of_rank[rank]

    # penalty parameters (reading Q20)
    t_hi = 10.0 if cfg["t_hi"] == "ten" else float(-(-n_items // cfg["C"]))
    t = stream_u01(seed, _S_T, K) * t_hi
    if cfg["vw"] == "unit":
        v = stream_u01(seed, _S_V, K)
        w = stream_u01(seed, _S_W, K)
    else:  # log-uniform 1e-3 .. 1e3
        v = 10.0 ** (stream_u01(seed, _S_V, K) * 6.0 - 3.0)
        w = 10.0 ** (stream_u01(seed, _S_W, K) * 6.0 - 3.0)
    return Problem(n_aisles=NA, slots_per_side=S, slot_pitch=1, aisle_spacing=3, depot_aisle=0,
                   sku_loc=sku_loc.astype(np.int32), sku_class=sku_class.astype(np.int32),
                   n_classes=K, order_ptr=order_ptr.astype(np.int32),
                   item_sku=item_sku.astype(np.int32), cart_capacity=cfg["C"], t=t, v=v, w=w)


def make_workload(name: str, seed: int = 0, **override) -> Workload:
    cfg = dict(CONFIGS[name], **override)
    pb = make_problem(name, seed, **override)
    return Workload(name=name, problem=pb, n_cand=cfg["n_cand"], seed=seed,
                    window=cfg.get("window", 0), stride=cfg.get("stride", 0),
                    n_iter=cfg.get("n_iter", 0))


# ---- candidate permutations (reading Q21): random keys, stable argsort ----------------------
def _perm_key_seed(seed: int) -> int:
    return int(_sub_seed(seed, _S_PERM))


def perm_rows(seed: int, n_orders: int, rows) -> np.ndarray:
    """Candidate permutations for the given candidate indices: int32 [len(rows)][n_orders].
    key(c,pos) = splitmix64(perm_seed ^ (c*n_orders+pos)) >> 1; pi_c = stable argsort."""
    rows = np.asarray(rows, dtype=np.uint64)
    ks = np.uint64(_perm_key_seed(seed))
    with np.errstate(over="ignore"):
        ctr = rows[:, None] * np.uint64(n_orders) + np.arange(n_orders, dtype=np.uint64)[None, :]
    keys = splitmix64(ks ^ ctr) >> np.uint64(1)
    return np.argsort(keys, axis=1, kind="stable").astype(np.int32)


def perms(seed: int, n_orders: int, n_cand: int) -> np.ndarray:
    out = np.empty((n_cand, n_orders), dtype=np.int32)
    step = max(1, (1 << 22) // max(n_orders, 1))
    for lo in range(0, n_cand, step):
        hi = min(n_cand, lo + step)
        out[lo:hi] = perm_rows(seed, n_orders, np.arange(lo, hi))
    return out


def base_perm(seed: int, n_orders: int) -> np.ndarray:
    """The single base sequence of the neighbourhood config."""
    return _shuffle(seed, _S_BASE, n_orders).astype(np.int32)


def perms_torch(seed: int, n_orders: int, lo: int, hi: int, device):
    """Same rows as perm_rows(seed, n_orders, range(lo, hi)), generated on `device` with torch
    integer ops (int64 wrap-around arithmetic, logical shifts via masks). Used to materialise
    the 5.24 GB stress candidate set directly in HBM."""
    import torch

    def s64(x):  # uint64 constant -> the int64 with the same bits
        x &= _M64
        return x - (1 << 64) if x >= (1 << 63) else x

    def lsr(z, k):
        return (z >> k) & ((1 << (64 - k)) - 1)

    c = torch.arange(lo, hi, device=device, dtype=torch.int64)[:, None]
    pos = torch.arange(n_orders, device=device, dtype=torch.int64)[None, :]
    z = (c * n_orders + pos) ^ s64(_perm_key_seed(seed))
    z = z + s64(_GAMMA)
    z = (z ^ lsr(z, 30)) * s64(_MUL1)
    z = (z ^ lsr(z, 27)) * s64(_MUL2)
    z = z ^ lsr(z, 31)
    keys = lsr(z, 1)
    return torch.argsort(keys, dim=1, stable=True).to(torch.int32)
