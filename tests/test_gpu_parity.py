"""GPU parity: the CUDA path (through the C-ABI binding) against the oracle, element by element
on the same seeded inputs. Bars (BASELINE.json north_star): bit-exact batch assignment, route
distances, responses and argmin index; fp64 penalty / objective within 1e-9 relative (the
canonical summation order of D6 makes them bit-identical in practice, which is also asserted
where the argmin depends on it)."""
import os

import numpy as np
import pytest

import oracle
from paper_2110_13693_b200 import workloads as W

pytestmark = pytest.mark.gpu

RTOL = 1e-9  # north_star: "within 1e-9 relative error for the fp64 penalty and total objective"


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


class force_general:
    """Route non-detail calls through the general walker instead of the tuned K1/K2/K3 path."""
    def __init__(self, ctx):
        self.ctx = ctx
    def __enter__(self):
        from paper_2110_13693_b200 import whp
        self.ctx.debug_set(whp.DEBUG_FORCE_GENERAL, 1)
    def __exit__(self, *a):
        from paper_2110_13693_b200 import whp
        self.ctx.debug_set(whp.DEBUG_FORCE_GENERAL, -1)


def gpu_eval(torch, ctx, perms_dev, detail=False):
    n = perms_dev.shape[0]
    dev = perms_dev.device
    out = {
        "dist": torch.full((n,), -1, dtype=torch.int64, device=dev),
        "penalty": torch.zeros(n, dtype=torch.float64, device=dev),
        "obj": torch.zeros(n, dtype=torch.float64, device=dev),
        "n_batches": torch.zeros(n, dtype=torch.int32, device=dev),
        "batch_hash": torch.zeros(n, dtype=torch.int64, device=dev),
    }
    if detail:
        out["batch_of_pos"] = torch.full((n, ctx.n_orders), -1, dtype=torch.int32, device=dev)
        out["n_distinct"] = torch.zeros(n, dtype=torch.int32, device=dev)
        out["resp"] = torch.zeros((n, ctx.n_classes), dtype=torch.int32, device=dev)
    ctx.eval_candidates(perms_dev, **out)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["batch_hash"] = res["batch_hash"].view(np.uint64)
    return res, out


def assert_parity(got, ref, pb, detail=False):
    assert np.array_equal(got["dist"], ref["dist"])
    assert np.array_equal(got["n_batches"], ref["n_batches"])
    assert np.array_equal(got["batch_hash"], ref["batch_hash"])
    # Q13: tolerance denominator for phi is max(|ref|, sum|term|, 1); sum|term| >= |ref|
    assert np.all(np.abs(got["penalty"] - ref["penalty"]) <= RTOL * np.maximum(np.abs(ref["penalty"]), 1.0))
    assert np.all(np.abs(got["obj"] - ref["obj"]) <= RTOL * np.abs(ref["obj"]))
    # canonical summation order (D6) => identical bits, which makes the argmin exact
    assert np.array_equal(got["penalty"], ref["penalty"])
    assert np.array_equal(got["obj"], ref["obj"])
    if detail:
        assert np.array_equal(got["batch_of_pos"], ref["batch_of_pos"])
        assert np.array_equal(got["resp"], ref["resp"])
        assert np.array_equal(got["n_distinct"], ref["n_distinct"])


def gpu_argmin(torch, ctx, obj_dev):
    idx = torch.full((1,), -7, dtype=torch.int64, device=obj_dev.device)
    val = torch.zeros(1, dtype=torch.float64, device=obj_dev.device)
    ctx.argmin(obj_dev, idx, val)
    torch.cuda.synchronize()
    return int(idx.item()), float(val.item())


# ---- configs 1 and 2: every candidate, every output --------------------------------------------
@pytest.mark.parametrize("name", ["tiny", "mid"])
def test_all_candidates_full_detail(torch_cuda, name):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload(name)
    pb = wl.problem
    perms = W.perms(wl.seed, pb.n_orders, wl.n_cand)
    ctx = whp.Context.from_problem(pb)
    got, dev = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda(), detail=True)
    ref = oracle.eval_candidates(pb, perms, detail=True)
    assert_parity(got, ref, pb, detail=True)
    # the timed path (no detail outputs) must give the same numbers
    got2, dev2 = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda(), detail=False)
    assert_parity(got2, ref, pb)
    with force_general(ctx):
        got3, _ = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda(), detail=False)
        # resp / batch_of_pos without n_distinct: the general kernel without its distinct-location scan
        resp_g = torch.full((wl.n_cand, pb.n_classes), -1, dtype=torch.int32, device="cuda")
        bop_g = torch.full((wl.n_cand, pb.n_orders), -1, dtype=torch.int32, device="cuda")
        ctx.eval_candidates(torch.from_numpy(perms).cuda(), resp=resp_g, batch_of_pos=bop_g)
        torch.cuda.synchronize()
    assert_parity(got3, ref, pb)
    assert np.array_equal(resp_g.cpu().numpy(), ref["resp"])
    assert np.array_equal(bop_g.cpu().numpy(), ref["batch_of_pos"])
    # responses alone come from the tuned path's vertical counters
    resp = torch.full((wl.n_cand, pb.n_classes), -1, dtype=torch.int32, device="cuda")
    ctx.eval_candidates(torch.from_numpy(perms).cuda(), resp=resp)
    torch.cuda.synchronize()
    assert np.array_equal(resp.cpu().numpy(), ref["resp"])
    i, v = gpu_argmin(torch, ctx, dev2["obj"])
    assert i == oracle.argmin(ref["obj"]) and v == ref["obj"][i]
    ctx.close()


def test_golden_examples_on_gpu(torch_cuda, golden):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    from test_oracle_pins import _golden_problem
    pb = _golden_problem(golden)
    ctx = whp.Context.from_problem(pb)
    perms = np.array([p["perm"] for p in golden["plans"]], np.int32)
    got, _ = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda(), detail=True)
    for i, ex in enumerate(golden["plans"]):
        assert got["batch_of_pos"][i].tolist() == ex["batch_of_pos"]
        assert int(got["dist"][i]) == ex["dist"] and got["resp"][i].tolist() == ex["resp"]
        assert got["penalty"][i] == ex["penalty"] and got["obj"][i] == ex["obj"]
        assert int(got["batch_hash"][i]) == ex["batch_hash"]
    assert int(got["n_distinct"][0]) == golden["plans"][0]["n_distinct"]
    # E6 through the swap evaluator
    e4, e6 = golden["plans"][0], golden["plans"][2]
    s, Wn = e6["window"]
    nn = Wn * (Wn - 1) // 2
    d = torch.zeros(nn, dtype=torch.int64, device="cuda")
    o = torch.zeros(nn, dtype=torch.float64, device="cuda")
    ctx.eval_swaps(torch.tensor(e4["perm"], dtype=torch.int32, device="cuda"), s, Wn, d, o)
    torch.cuda.synchronize()
    assert int(d[e6["neighbour_index"]]) == e6["dist"] and float(o[e6["neighbour_index"]]) == e6["obj"]
    ctx.close()


# ---- config 3 at full size, in the launch configuration bench.py times --------------------------
def test_paper_scale_full_launch_sampled_oracle(torch_cuda):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload("paper")
    pb = wl.problem
    ctx = whp.Context.from_problem(pb)
    perms_dev = W.perms_torch(wl.seed, pb.n_orders, 0, wl.n_cand, "cuda")
    assert ctx.validate_perms(perms_dev) == 0
    got, dev = gpu_eval(torch, ctx, perms_dev)  # all 16,384 candidates, timed-path outputs
    rows = np.unique(np.concatenate([np.arange(0, 96), np.arange(wl.n_cand - 96, wl.n_cand),
                                     (W.stream_u64(7, 1, 320) % np.uint64(wl.n_cand)).astype(np.int64)]))
    sample = W.perm_rows(wl.seed, pb.n_orders, rows)
    assert np.array_equal(sample, perms_dev[torch.from_numpy(rows).cuda()].cpu().numpy())
    ref = oracle.eval_candidates(pb, sample, detail=True)
    assert_parity({k: v[rows] for k, v in got.items()}, ref, pb)
    # detail outputs on the sampled rows
    gd, _ = gpu_eval(torch, ctx, torch.from_numpy(sample).cuda(), detail=True)
    assert_parity(gd, ref, pb, detail=True)
    # properties that hold for every candidate at any size
    q = np.diff(pb.order_ptr)
    assert np.all(got["n_batches"] >= -(-pb.n_items // pb.cart_capacity))
    assert np.all(got["dist"] > 0) and np.all(got["obj"] == got["dist"] + got["penalty"])
    # argmin over all candidates: index equals numpy's first minimum of the GPU objective,
    # and the winner's objective equals the oracle's for that row
    i, v = gpu_argmin(torch, ctx, dev["obj"])
    assert i == int(np.argmin(got["obj"])) and v == got["obj"][i]
    win = oracle.eval_candidates(pb, W.perm_rows(wl.seed, pb.n_orders, [i]))
    assert win["obj"][0] == v
    ctx.close()


def test_paper_scale_legsum_and_nhatc_sampled_oracle(torch_cuda):
    """NEXT-1 / NEXT-2 at the size bench.py times: leg sums of all 16,384 plans checked on
    sampled rows; two NHATC outer iterations over the first 2,048 plans against the oracle's loop."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload("paper")
    pb = wl.problem
    ctx = whp.Context.from_problem(pb)
    perms_dev = W.perms_torch(wl.seed, pb.n_orders, 0, wl.n_cand, "cuda")
    leg = torch.full((wl.n_cand,), -1, dtype=torch.int64, device="cuda")
    ctx.eval_legsum(perms_dev, leg)
    torch.cuda.synchronize()
    rows = np.unique(np.concatenate([np.arange(0, 40), np.arange(wl.n_cand - 40, wl.n_cand),
                                     (W.stream_u64(8, 1, 120) % np.uint64(wl.n_cand)).astype(np.int64)]))
    sample = W.perm_rows(wl.seed, pb.n_orders, rows)
    assert np.array_equal(leg.cpu().numpy()[rows], oracle.eval_legsum(pb, sample))
    assert int(leg.min()) > 0
    n_sub, n_outer, beta = 2048, 2, 1.25
    sub = W.perm_rows(wl.seed, pb.n_orders, np.arange(n_sub))
    idx = torch.zeros(n_outer, dtype=torch.int64, device="cuda")
    obj = torch.zeros(n_outer, dtype=torch.float64, device="cuda")
    ctx.nhatc_solve(perms_dev[:n_sub], n_outer, beta, idx, None, obj)
    torch.cuda.synchronize()
    ref = oracle.nhatc_loop(pb, sub, n_outer, beta)
    assert np.array_equal(idx.cpu().numpy(), ref["idx"]) and np.array_equal(obj.cpu().numpy(), ref["obj"])
    t, v, w = ctx.get_penalty()
    assert np.array_equal(v, ref["v"]) and np.array_equal(w, ref["w"])
    ctx.close()


# ---- config 5 (stress): 65,536 candidates generated in HBM, oracle on sampled rows ---------------
def test_stress_full_size_sampled_oracle(torch_cuda):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload("stress")
    pb = wl.problem
    ctx = whp.Context.from_problem(pb)
    n = pb.n_orders
    perms_dev = torch.empty((wl.n_cand, n), dtype=torch.int32, device="cuda")
    step = 4096
    for lo in range(0, wl.n_cand, step):
        perms_dev[lo:lo + step] = W.perms_torch(wl.seed, n, lo, lo + step, "cuda")
    got, dev = gpu_eval(torch, ctx, perms_dev)
    rows = np.unique(np.concatenate([[0, 1, wl.n_cand - 1],
                                     (W.stream_u64(9, 2, 45) % np.uint64(wl.n_cand)).astype(np.int64)]))
    sample = W.perm_rows(wl.seed, n, rows)
    assert np.array_equal(sample, perms_dev[torch.from_numpy(rows).cuda()].cpu().numpy())
    ref = oracle.eval_candidates(pb, sample, detail=True)
    assert_parity({k: v[rows] for k, v in got.items()}, ref, pb)
    gd, _ = gpu_eval(torch, ctx, torch.from_numpy(sample[:8]).cuda(), detail=True)
    assert_parity(gd, {k: v[:8] for k, v in ref.items()}, pb, detail=True)
    i, v = gpu_argmin(torch, ctx, dev["obj"])
    assert i == int(np.argmin(got["obj"])) and v == got["obj"][i]
    win = oracle.eval_candidates(pb, W.perm_rows(wl.seed, n, [i]))
    assert win["obj"][0] == v and win["dist"][0] == got["dist"][i]
    # NEXT-2 at this size: the pick table (265 KB) does not fit shared memory, so the leg-sum
    # kernel gathers it through L2 like the set kernel does
    head = W.perm_rows(wl.seed, n, np.arange(40))
    leg = torch.full((40,), -1, dtype=torch.int64, device="cuda")
    ctx.eval_legsum(perms_dev[:40], leg)
    torch.cuda.synchronize()
    assert np.array_equal(leg.cpu().numpy(), oracle.eval_legsum(pb, head))
    # NEXT-1 at this size (K = 32: one class word), 3 outer iterations over 256 plans
    hist = oracle.nhatc_loop(pb, W.perm_rows(wl.seed, n, np.arange(256)), 3, 1.5)
    idx_h = torch.zeros(3, dtype=torch.int64, device="cuda")
    ctx.nhatc_solve(perms_dev[:256], 3, 1.5, idx_h)
    t2, v2, w2 = ctx.get_penalty()
    assert np.array_equal(idx_h.cpu().numpy(), hist["idx"])
    assert np.array_equal(v2, hist["v"]) and np.array_equal(w2, hist["w"])
    ctx.close()


BIG_TABLES = [
    # pick tables beyond shared memory (the tuned path gathers them through L1 / L2)
    dict(NA=400, S=250, K=32, n_skus=20000, n_orders=16000, qmax=5, C=40),              # stress-like
    dict(NA=400, S=250, K=200, n_skus=20000, n_orders=12000, qmax=7, C=30, depot=123),  # 7 class words
    dict(NA=1024, S=100, K=64, n_skus=9000, n_orders=30000, qmax=1, C=17, pitch=2),     # one-pick orders
    dict(NA=90, S=4095, K=256, n_skus=9000, n_orders=9000, qmax=13, C=64, spacing=9),   # many fours an order
    dict(NA=700, S=60, K=17, n_skus=30000, n_orders=10001, qmax=9, C=106, depot=699),   # largest cart, padded plans
    dict(NA=33, S=9, K=1, n_skus=500, n_orders=600, qmax=255, C=255),                   # 64 fours an order
    dict(NA=1024, S=4095, K=32, n_skus=60000, n_orders=50000, qmax=2, C=12, spacing=11), # ~6,500 carts a plan
]


@pytest.mark.parametrize("cfg", BIG_TABLES, ids=lambda c: "-".join(f"{k}{v}" for k, v in c.items()))
def test_tables_beyond_shared_memory_both_set_kernels(torch_cuda, cfg):
    """The four-aligned set kernel (default) and the pair-load variant (WHP_DEBUG_NO_FOURS) both
    equal the oracle, with every segment count, on candidate counts that leave warp tails."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = _random_problem(23, **cfg)
    ctx = whp.Context.from_problem(pb)
    perms = W.perm_rows(5, pb.n_orders, np.arange(37))
    ref = oracle.eval_candidates(pb, perms, detail=True)
    d_perms = torch.from_numpy(perms).cuda()
    for no_fours in (0, 1):
        ctx.debug_set(whp.DEBUG_NO_FOURS, no_fours)
        for seg in (-1, 8, 32):
            ctx.debug_set(whp.DEBUG_SEGMENTS, seg)
            got, _ = gpu_eval(torch, ctx, d_perms)
            assert_parity(got, ref, pb)
            resp = torch.zeros((37, pb.n_classes), dtype=torch.int32, device="cuda")
            ctx.eval_candidates(d_perms, resp=resp)
            torch.cuda.synchronize()
            assert np.array_equal(resp.cpu().numpy(), ref["resp"])
    ctx.debug_set(whp.DEBUG_SEGMENTS, -1)
    want = oracle.eval_legsum(pb, perms)
    for no_fours in (0, 1):  # the leg kernel has both layouts too
        ctx.debug_set(whp.DEBUG_NO_FOURS, no_fours)
        leg = torch.full((37,), -1, dtype=torch.int64, device="cuda")
        ctx.eval_legsum(d_perms, leg)
        torch.cuda.synchronize()
        assert np.array_equal(leg.cpu().numpy(), want)
    ctx.debug_set(whp.DEBUG_NO_FOURS, -1)
    ctx.close()


def test_more_orders_than_the_tuned_path_indexes(torch_cuda):
    """66,000 orders: positions no longer fit the 16-bit cursors, so evaluation, leg sums and the
    neighbourhood all take their general kernels (and the swap base pass runs without
    shared-memory tables)."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = _random_problem(4, NA=50, S=40, K=70, n_skus=3000, n_orders=66000, qmax=4, C=9)
    ctx = whp.Context.from_problem(pb)
    perms = W.perm_rows(8, pb.n_orders, np.arange(6))
    got, _ = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda(), detail=True)
    ref = oracle.eval_candidates(pb, perms, detail=True)
    assert_parity(got, ref, pb, detail=True)
    leg = torch.zeros(6, dtype=torch.int64, device="cuda")
    ctx.eval_legsum(torch.from_numpy(perms).cuda(), leg)
    torch.cuda.synchronize()
    assert np.array_equal(leg.cpu().numpy(), oracle.eval_legsum(pb, perms))
    s, Wn = 40000, 9
    d = torch.zeros(Wn * (Wn - 1) // 2, dtype=torch.int64, device="cuda")
    o = torch.zeros(Wn * (Wn - 1) // 2, dtype=torch.float64, device="cuda")
    ctx.eval_swaps(torch.from_numpy(perms[0]).cuda(), s, Wn, d, o)
    torch.cuda.synchronize()
    rs = oracle.eval_swaps(pb, perms[0], s, Wn)
    assert np.array_equal(d.cpu().numpy(), rs["dist"]) and np.array_equal(o.cpu().numpy(), rs["obj"])
    ctx.close()


# ---- edge cases ----------------------------------------------------------------------------------
def _random_problem(seed, NA, S, K, n_skus, n_orders, qmax, C, depot=0, pitch=1, spacing=3):
    rng = np.random.default_rng(seed)
    q = rng.integers(1, qmax + 1, size=n_orders)
    ptr = np.concatenate([[0], np.cumsum(q)]).astype(np.int32)
    return W.Problem(
        n_aisles=NA, slots_per_side=S, slot_pitch=pitch, aisle_spacing=spacing, depot_aisle=depot,
        sku_loc=rng.integers(0, 2 * NA * S, size=n_skus).astype(np.int32),
        sku_class=rng.integers(0, K, size=n_skus).astype(np.int32), n_classes=K, order_ptr=ptr,
        item_sku=rng.integers(0, n_skus, size=int(ptr[-1])).astype(np.int32), cart_capacity=C,
        t=rng.uniform(0, 20, K), v=rng.uniform(-1, 1, K), w=rng.uniform(0, 2, K))


EDGE = [
    dict(NA=1, S=1, K=1, n_skus=1, n_orders=1, qmax=1, C=1),            # the smallest problem
    dict(NA=1, S=7, K=1, n_skus=5, n_orders=33, qmax=3, C=3),           # one aisle, one class
    dict(NA=5, S=9, K=3, n_skus=30, n_orders=31, qmax=4, C=4),          # ragged tile (31)
    dict(NA=5, S=9, K=3, n_skus=30, n_orders=32, qmax=4, C=1000),       # one batch holds all
    dict(NA=37, S=11, K=33, n_skus=200, n_orders=97, qmax=1, C=1),      # every order is a batch
    dict(NA=64, S=20, K=64, n_skus=500, n_orders=257, qmax=6, C=6, depot=20),   # depot mid-floor
    dict(NA=1024, S=30, K=256, n_skus=5000, n_orders=1000, qmax=12, C=40, depot=1023, pitch=3, spacing=7),
    dict(NA=400, S=4095, K=200, n_skus=3000, n_orders=333, qmax=255, C=600),    # limits: q, slots
    dict(NA=33, S=17, K=40, n_skus=100, n_orders=129, qmax=5, C=70),    # batches longer than a tile
    # multiples of 4 orders: these run the tuned K1/K2/K3 path
    dict(NA=1, S=1, K=1, n_skus=1, n_orders=4, qmax=1, C=1),
    dict(NA=5, S=9, K=3, n_skus=30, n_orders=32, qmax=4, C=4),
    dict(NA=17, S=9, K=255, n_skus=300, n_orders=260, qmax=9, C=9, depot=5, pitch=2),
    dict(NA=1024, S=30, K=256, n_skus=5000, n_orders=1000, qmax=12, C=40, depot=1023, pitch=3, spacing=7),
    dict(NA=1024, S=30, K=256, n_skus=5000, n_orders=1000, qmax=12, C=40),
    dict(NA=400, S=4095, K=200, n_skus=3000, n_orders=332, qmax=255, C=600),
    dict(NA=40, S=50, K=20, n_skus=900, n_orders=2000, qmax=2, C=2),    # ~1,500 batches per plan
    dict(NA=40, S=50, K=20, n_skus=900, n_orders=64, qmax=3, C=100000), # one batch, huge cart
    dict(NA=60, S=30, K=90, n_skus=700, n_orders=400, qmax=7, C=106),   # largest cart of the tuned path
    dict(NA=60, S=30, K=90, n_skus=700, n_orders=403, qmax=7, C=65),    # 16-chunk cursor ring
    dict(NA=60, S=30, K=90, n_skus=700, n_orders=401, qmax=7, C=107),   # one item more: general path
]


@pytest.mark.parametrize("cfg", EDGE, ids=lambda c: "-".join(f"{k}{v}" for k, v in c.items()))
def test_edge_cases(torch_cuda, cfg):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = _random_problem(11, **cfg)
    ctx = whp.Context.from_problem(pb)
    perms = W.perm_rows(3, pb.n_orders, np.arange(70))
    got, dev = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda(), detail=True)
    ref = oracle.eval_candidates(pb, perms, detail=True)
    assert_parity(got, ref, pb, detail=True)
    got2, dev2 = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda())
    assert_parity(got2, ref, pb)
    with force_general(ctx):
        got3, _ = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda())
    assert_parity(got3, ref, pb)
    for seg in ("1", "2", "32"):  # segment counts of the tuned path (ignored when not legal)
        ctx.debug_set(whp.DEBUG_SEGMENTS, int(seg))
        got4, _ = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda())
        ctx.debug_set(whp.DEBUG_SEGMENTS, -1)
        assert_parity(got4, ref, pb)
    i, v = gpu_argmin(torch, ctx, dev2["obj"])
    assert i == oracle.argmin(ref["obj"])
    ctx.close()


@pytest.mark.parametrize("n_orders", [5, 8, 28, 31, 33, 36, 60, 63, 64, 65, 68, 96, 97, 100, 128, 130,
                                      132, 192, 195, 196])
@pytest.mark.parametrize("n_cand", [1, 33])
def test_tuned_path_word_and_warp_tails(torch_cuda, n_orders, n_cand):
    """K1 streams 32 plans x 32 positions per tile: every combination of full / partial last
    word, odd / even number of words and a partial last warp of plans must agree with the
    oracle (plan lengths that are no multiple of 4 go through a padded copy)."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = _random_problem(5, NA=70, S=12, K=70, n_skus=400, n_orders=n_orders, qmax=5, C=11, depot=3)
    ctx = whp.Context.from_problem(pb)
    perms = W.perm_rows(7, pb.n_orders, np.arange(n_cand))
    got, dev = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda())
    ref = oracle.eval_candidates(pb, perms, detail=True)
    assert_parity(got, ref, pb)
    for kw in (2, 4):  # K1 blocks of two / four warps sharing the order table
        ctx.debug_set(whp.DEBUG_K1_WARPS, kw)
        got_k, _ = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda())
        assert_parity(got_k, ref, pb)
    ctx.debug_set(whp.DEBUG_K1_WARPS, -1)
    # batch_of_pos alone stays on the tuned path (derived from K1's boundary mask)
    bop = torch.full((n_cand, pb.n_orders), -1, dtype=torch.int32, device="cuda")
    d2 = torch.zeros(n_cand, dtype=torch.int64, device="cuda")
    ctx.eval_candidates(torch.from_numpy(perms).cuda(), dist=d2, batch_of_pos=bop)
    torch.cuda.synchronize()
    assert np.array_equal(bop.cpu().numpy(), ref["batch_of_pos"])
    assert np.array_equal(d2.cpu().numpy(), ref["dist"])
    ctx.close()


@pytest.mark.parametrize("name,n_cand", [("tiny", 37), ("mid", 100)])
def test_outputs_stay_inside_their_buffers(torch_cuda, name, n_cand):
    """Every caller buffer sits between guard words; no kernel (tuned path, general path, swaps,
    argmin) may touch a guard (compute-sanitizer is not available on the GPU pool)."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem(name)
    ctx = whp.Context.from_problem(pb)
    G = 64

    def guarded(shape, dtype):
        n = int(np.prod(shape))
        buf = torch.full((n + 2 * G,), 0x5A, dtype=dtype, device="cuda")
        return buf, buf[G:G + n].view(*shape)

    perms_np = W.perms(1, pb.n_orders, n_cand)
    pbuf, perms = guarded((n_cand, pb.n_orders), torch.int32)
    perms.copy_(torch.from_numpy(perms_np))
    bufs = {}
    for key, shape, dt in (("dist", (n_cand,), torch.int64), ("penalty", (n_cand,), torch.float64),
                           ("obj", (n_cand,), torch.float64), ("n_batches", (n_cand,), torch.int32),
                           ("batch_hash", (n_cand,), torch.int64),
                           ("resp", (n_cand, pb.n_classes), torch.int32),
                           ("batch_of_pos", (n_cand, pb.n_orders), torch.int32),
                           ("n_distinct", (n_cand,), torch.int32)):
        bufs[key] = guarded(shape, dt)
    tuned = {k: v[1] for k, v in bufs.items() if k not in ("batch_of_pos", "n_distinct")}
    ctx.eval_candidates(perms, **tuned)
    ctx.eval_candidates(perms, **{k: v[1] for k, v in bufs.items()})
    Wn = min(12, pb.n_orders)
    nn = Wn * (Wn - 1) // 2
    sd, so = guarded((nn,), torch.int64), guarded((nn,), torch.float64)
    ibuf, idx = guarded((1,), torch.int64)
    base_buf, base = guarded((pb.n_orders,), torch.int32)
    base.copy_(perms[0])
    ctx.eval_swaps(base, 1, Wn, sd[1], so[1])
    ctx.argmin(so[1], idx)
    ctx.apply_swap(base, 1, Wn, idx)
    torch.cuda.synchronize()
    for name_, (buf, view) in list(bufs.items()) + [("sd", sd), ("so", so), ("idx", (ibuf, idx)),
                                                     ("base", (base_buf, base)), ("perms", (pbuf, perms))]:
        guard = torch.full((G,), 0x5A, dtype=buf.dtype, device="cuda")
        assert torch.equal(buf[:G], guard) and torch.equal(buf[-G:], guard), name_
    assert np.array_equal(perms.cpu().numpy(), perms_np)
    ref = oracle.eval_candidates(pb, perms_np, detail=True)
    assert np.array_equal(bufs["dist"][1].cpu().numpy(), ref["dist"])
    assert np.array_equal(bufs["resp"][1].cpu().numpy(), ref["resp"])
    ctx.close()


def test_unaligned_permutation_buffer(torch_cuda):
    """A permutation matrix that starts 4 bytes off a 16-byte boundary cannot be described by a
    TMA tensor map: the call must still be right (the plans go through an aligned copy)."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid")
    ctx = whp.Context.from_problem(pb)
    perms_np = W.perms(2, pb.n_orders, 50)
    buf = torch.zeros(50 * pb.n_orders + 8, dtype=torch.int32, device="cuda")
    perms = buf[1:1 + 50 * pb.n_orders].view(50, pb.n_orders)
    assert perms.data_ptr() % 16 == 4
    perms.copy_(torch.from_numpy(perms_np))
    got, _ = gpu_eval(torch, ctx, perms)
    assert_parity(got, oracle.eval_candidates(pb, perms_np), pb)
    ctx.close()


@pytest.mark.parametrize("name,n_cand", [("tiny", 64), ("mid", 300)])
def test_legsum_matches_oracle(torch_cuda, name, n_cand):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem(name)
    ctx = whp.Context.from_problem(pb)
    perms = W.perms(0, pb.n_orders, n_cand)
    out = torch.full((n_cand,), -1, dtype=torch.int64, device="cuda")
    ctx.eval_legsum(torch.from_numpy(perms).cuda(), out)
    torch.cuda.synchronize()
    ref = oracle.eval_legsum(pb, perms)
    assert np.array_equal(out.cpu().numpy(), ref)
    out.fill_(-1)
    with force_general(ctx):  # the warp-per-plan kernel
        ctx.eval_legsum(torch.from_numpy(perms).cuda(), out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref)
    ctx.close()


@pytest.mark.parametrize("cfg", EDGE, ids=lambda c: "-".join(f"{k}{v}" for k, v in c.items()))
def test_legsum_edge_cases(torch_cuda, cfg):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = _random_problem(13, **cfg)
    ctx = whp.Context.from_problem(pb)
    perms = W.perm_rows(5, pb.n_orders, np.arange(40))
    out = torch.full((40,), -1, dtype=torch.int64, device="cuda")
    ctx.eval_legsum(torch.from_numpy(perms).cuda(), out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), oracle.eval_legsum(pb, perms))
    ctx.close()


@pytest.mark.parametrize("name,k,Z,iters", [("tiny", 4, 1, 5), ("mid", 10, 2, 8), ("paper", 50, 4, 12),
                                            ("mid", 7, 3, 0)])
def test_kmeans_slotting_matches_oracle(torch_cuda, name, k, Z, iters):
    """NEXT-3 (reading N3): frequencies, assignment, centroids and the slotting are bit-identical
    to the oracle (integer sums, one fp64 division per centroid); the layout it produces feeds
    whp_create_layout and the evaluator agrees with the oracle on it."""
    torch = torch_cuda
    import copy
    from paper_2110_13693_b200 import whp
    pb = W.make_problem(name)
    got = whp.kmeans_slotting(pb.n_aisles, pb.slots_per_side, pb.depot_aisle, pb.n_skus,
                              pb.item_sku, k, Z, iters)
    ref = oracle.kmeans_slotting(pb, pb.n_skus, pb.item_sku, k, Z, iters)
    for key in ("assign", "centroids", "sku_loc", "sku_class"):
        assert np.array_equal(got[key], ref[key]), key
    pb2 = copy.copy(pb)
    pb2.sku_loc, pb2.sku_class, pb2.n_classes = got["sku_loc"], got["sku_class"], k * Z
    rng = np.random.default_rng(0)
    pb2.t, pb2.v, pb2.w = rng.uniform(0, 9, k * Z), rng.uniform(0, 1, k * Z), rng.uniform(0, 1, k * Z)
    ctx = whp.Context.from_problem(pb2)
    perms = W.perms(0, pb.n_orders, 24)
    g, _ = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda())
    assert_parity(g, oracle.eval_candidates(pb2, perms), pb2)
    ctx.close()


def test_kmeans_slotting_hand_worked_and_errors(torch_cuda):
    from paper_2110_13693_b200 import whp
    items = [0] * 5 + [1] + [2] + [3] * 6 + [4] + [5] * 5
    out = whp.kmeans_slotting(3, 2, 0, 6, items, 2, 1, 3)
    assert out["assign"].tolist() == [1, 0, 0, 1, 0, 1]
    assert out["centroids"].tolist() == [1.0, 16.0 / 3.0]
    assert out["sku_loc"].tolist() == [0, 3, 4, 2, 6, 1]
    with pytest.raises(whp.WhpError):
        whp.kmeans_slotting(1, 2, 0, 6, items, 2, 1, 3)       # 6 SKUs, 4 locations
    with pytest.raises(whp.WhpError):
        whp.kmeans_slotting(3, 2, 0, 6, items + [6], 2, 1, 3)  # SKU id out of range


def _adversarial_perm(pb):
    """A plan with (nearly) as many carts as possible: every cart is filled with small orders just
    far enough that the next, large order does not fit — the situation the static bound on the
    batch count (and with it the number of counter planes of K2) has to cover."""
    q = np.diff(pb.order_ptr)
    C = pb.cart_capacity
    big = list(np.argsort(-q, kind="stable"))          # large orders open the carts
    small = list(np.argsort(q, kind="stable"))         # small orders fill them
    used = np.zeros(len(q), bool)
    perm, load, bi, si = [], 0, 0, 0
    while len(perm) < len(q):
        while bi < len(big) and used[big[bi]]:
            bi += 1
        while si < len(small) and used[small[si]]:
            si += 1
        if bi >= len(big):
            break
        b = big[bi]
        if load + q[b] > C or si >= len(small) or small[si] == b:
            perm.append(b); used[b] = True                # opens a new cart (or nothing else left)
            load = q[b] if load + q[b] > C else load + q[b]
        else:
            s_ = small[si]
            perm.append(s_); used[s_] = True
            load = q[s_] if load + q[s_] > C else load + q[s_]
    return np.array(perm, dtype=np.int32)


@pytest.mark.parametrize("name", ["mid", "paper"])
def test_many_cart_plans_stay_within_the_counter_planes(torch_cuda, name):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem(name)
    adv = _adversarial_perm(pb)
    assert sorted(adv.tolist()) == list(range(pb.n_orders))
    perms = np.stack([adv, adv[::-1].copy(), W.perm_rows(0, pb.n_orders, [0])[0]] * 11).astype(np.int32)
    ctx = whp.Context.from_problem(pb)
    got, _ = gpu_eval(torch, ctx, torch.from_numpy(perms).cuda(), detail=False)
    ref = oracle.eval_candidates(pb, perms)
    assert ref["n_batches"][0] > 1.1 * ref["n_batches"][2]        # really more carts than a random plan
    assert_parity(got, ref, pb)
    ctx.close()


def test_batch_count_bound_holds_for_every_permutation(torch_cuda):
    """whp_max_batches sizes K2's counters: it must bound the cart count of EVERY plan. Checked
    exhaustively (all 5,040 orders of 7 orders, several random problems) and on the adversarial
    plans of the named workloads; it is also reasonably tight."""
    import itertools
    from paper_2110_13693_b200 import whp
    rng = np.random.default_rng(9)
    for trial in range(6):
        C = int(rng.integers(3, 9))
        q = rng.integers(1, min(C, 5) + 1, size=7)
        ptr = np.concatenate([[0], np.cumsum(q)]).astype(np.int32)
        pb = W.Problem(n_aisles=3, slots_per_side=4, slot_pitch=1, aisle_spacing=2, depot_aisle=0,
                       sku_loc=np.arange(10, dtype=np.int32), sku_class=np.zeros(10, np.int32),
                       n_classes=1, order_ptr=ptr,
                       item_sku=rng.integers(0, 10, size=int(ptr[-1])).astype(np.int32),
                       cart_capacity=C, t=np.zeros(1), v=np.zeros(1), w=np.zeros(1))
        ctx = whp.Context.from_problem(pb)
        bound = ctx.max_batches()
        perms = np.array(list(itertools.permutations(range(7))), dtype=np.int32)
        nb = oracle.eval_candidates(pb, perms)["n_batches"]
        assert nb.max() <= bound <= nb.max() + 1, (q, C, nb.max(), bound)
        ctx.close()
    for name in ("mid", "paper", "stress"):
        pb = W.make_problem(name)
        ctx = whp.Context.from_problem(pb)
        adv = _adversarial_perm(pb)
        nb = oracle.eval_candidates(pb, adv)["n_batches"][0]
        assert nb <= ctx.max_batches() <= 1.12 * nb
        ctx.close()


def test_api_errors_and_nullable_outputs(torch_cuda):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("tiny")
    ctx = whp.Context(pb.n_aisles, pb.slots_per_side, pb.slot_pitch, pb.aisle_spacing,
                      pb.depot_aisle, pb.sku_loc, pb.sku_class, pb.n_classes)
    perms = torch.from_numpy(W.perms(0, pb.n_orders, 4)).cuda()
    obj = torch.zeros(4, dtype=torch.float64, device="cuda")
    ctx.n_orders = pb.n_orders
    with pytest.raises(whp.WhpError) as e:
        ctx.eval_candidates(perms, obj=obj)  # before load_orders
    assert e.value.status == whp.ERR_STATE
    with pytest.raises(whp.WhpError) as e:
        ctx.load_orders(pb.order_ptr, pb.item_sku, 3)  # an order of 4 items, cart of 3
    assert e.value.status == whp.ERR_CAPACITY
    with pytest.raises(whp.WhpError) as e:
        ctx.load_orders(pb.order_ptr, pb.item_sku + 1000, 8)
    assert e.value.status == whp.ERR_OUT_OF_RANGE
    ctx.load_orders(pb.order_ptr, pb.item_sku, pb.cart_capacity)
    with pytest.raises(whp.WhpError) as e:
        ctx.eval_candidates(perms, obj=obj)  # before set_penalty
    assert e.value.status == whp.ERR_STATE
    with pytest.raises(whp.WhpError) as e:
        ctx.set_penalty(pb.t, pb.v * np.inf, pb.w)
    assert e.value.status == whp.ERR_OUT_OF_RANGE
    ctx.set_penalty(pb.t, pb.v, pb.w)
    ctx.eval_candidates(perms, obj=obj)  # only one output requested
    ctx.eval_candidates(perms[:0], obj=obj)  # empty input is a no-op
    torch.cuda.synchronize()
    ref = oracle.eval_candidates(pb, perms.cpu().numpy())
    assert np.array_equal(obj.cpu().numpy(), ref["obj"])
    with pytest.raises(whp.WhpError) as e:
        ctx.eval_swaps(perms[0], 0, 1, obj=obj)
    assert e.value.status == whp.ERR_INVALID_ARG
    with pytest.raises(whp.WhpError) as e:
        ctx.eval_swaps(perms[0], 15, 6, obj=torch.zeros(15, dtype=torch.float64, device="cuda"))
    assert e.value.status == whp.ERR_OUT_OF_RANGE
    bad = perms.clone()
    bad[2, 0] = bad[2, 1]
    assert ctx.validate_perms(bad) == 1 and ctx.validate_perms(perms) == 0
    # argmin: ties -> lowest index; single element; works on a non-default stream
    x = torch.tensor([3.0, 1.0, 2.0, 1.0, 1.0], dtype=torch.float64, device="cuda")
    s = torch.cuda.Stream()
    idx = torch.zeros(1, dtype=torch.int64, device="cuda")
    with torch.cuda.stream(s):
        ctx.argmin(x, idx)
    s.synchronize()
    assert int(idx) == 1
    ctx.argmin(x[:1], idx)
    torch.cuda.synchronize()
    assert int(idx) == 0
    big = torch.full((1 << 20,), 5.0, dtype=torch.float64, device="cuda")
    big[777777] = 4.0
    big[999999] = 4.0
    ctx.argmin(big, idx)
    torch.cuda.synchronize()
    assert int(idx) == 777777
    # replacing orders and penalty on a live context
    pb2 = _random_problem(5, 4, 10, 4, 40, 25, 3, 5)
    ctx.load_orders(pb2.order_ptr, pb2.item_sku, pb2.cart_capacity)
    ctx.set_penalty(pb2.t, pb2.v, pb2.w)
    pb2.sku_loc, pb2.sku_class = pb.sku_loc, pb.sku_class
    p2 = W.perms(1, pb2.n_orders, 6)
    got, _ = gpu_eval(torch, ctx, torch.from_numpy(p2).cuda())
    assert_parity(got, oracle.eval_candidates(pb2, p2), pb2)
    ctx.close()


def test_host_buffer_entry_point(torch_cuda):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload("mid")
    pb = wl.problem
    ctx = whp.Context.from_problem(pb)
    perms = W.perms(wl.seed, pb.n_orders, wl.n_cand)
    ref = oracle.eval_candidates(pb, perms)
    # pageable numpy buffers
    dist = np.zeros(wl.n_cand, np.int64)
    obj = np.zeros(wl.n_cand, np.float64)
    i, v = ctx.eval_candidates_host(perms, dist, obj)
    assert np.array_equal(dist, ref["dist"]) and np.array_equal(obj, ref["obj"])
    assert i == oracle.argmin(ref["obj"]) and v == ref["obj"][i]
    # pinned torch buffers
    pp = torch.from_numpy(perms).pin_memory()
    pd = torch.zeros(wl.n_cand, dtype=torch.int64).pin_memory()
    po = torch.zeros(wl.n_cand, dtype=torch.float64).pin_memory()
    i2, v2 = ctx.eval_candidates_host(pp, pd, po)
    assert (i2, v2) == (i, v) and np.array_equal(pd.numpy(), ref["dist"])
    assert np.array_equal(po.numpy(), ref["obj"])
    ctx.close()


# ---- host-buffer entry points (int32 and uint16 order ids) -------------------------------------------
@pytest.mark.parametrize("n_orders,n_cand", [(500, 700), (64, 33), (97, 5), (36, 1), (4000, 300), (130, 64)])
def test_host_entry_points_int32_and_uint16(torch_cuda, n_orders, n_cand):
    """whp_eval_candidates_host / _host16 (chunked copies overlapped with evaluation) equal the
    oracle; the 16-bit call runs K1 on 16-bit tiles (64 positions per tile row), including plan
    lengths that are no multiple of 8 (padded copy) and of 64 (partial last tile)."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    if n_orders == 4000:
        pb = W.make_problem("paper")
    elif n_orders == 500:
        pb = W.make_problem("mid")
    else:
        pb = _random_problem(9, NA=70, S=12, K=70, n_skus=400, n_orders=n_orders, qmax=5, C=11, depot=3)
    ctx = whp.Context.from_problem(pb)
    perms = W.perm_rows(3, pb.n_orders, np.arange(n_cand))
    ref = oracle.eval_candidates(pb, perms)
    for arr in (perms, perms.astype(np.uint16)):
        d, o = np.zeros(n_cand, np.int64), np.zeros(n_cand, np.float64)
        i, v = ctx.eval_candidates_host(np.ascontiguousarray(arr), d, o)
        assert np.array_equal(d, ref["dist"]) and np.array_equal(o, ref["obj"]), arr.dtype
        assert i == oracle.argmin(ref["obj"]) and v == ref["obj"][i]
    # pinned torch buffers, 16-bit ids as int16 bit patterns
    h16 = torch.from_numpy(perms.astype(np.uint16).view(np.int16)).pin_memory()
    hd = torch.zeros(n_cand, dtype=torch.int64).pin_memory()
    ho = torch.zeros(n_cand, dtype=torch.float64).pin_memory()
    i, v = ctx.eval_candidates_host(h16, hd, ho)
    assert np.array_equal(hd.numpy(), ref["dist"]) and np.array_equal(ho.numpy(), ref["obj"])
    ctx.close()


def test_host16_needs_a_tuned_path_shape(torch_cuda):
    from paper_2110_13693_b200 import whp
    pb = _random_problem(4, NA=50, S=40, K=70, n_skus=3000, n_orders=300, qmax=4, C=200)  # C > 106
    ctx = whp.Context.from_problem(pb)
    perms = W.perm_rows(8, pb.n_orders, np.arange(6))
    with pytest.raises(whp.WhpError) as e:
        ctx.eval_candidates_host(perms.astype(np.uint16), np.zeros(6, np.int64))
    assert e.value.status == whp.ERR_OUT_OF_RANGE
    d = np.zeros(6, np.int64)
    ctx.eval_candidates_host(perms, d)  # the int32 call takes any shape
    assert np.array_equal(d, oracle.eval_candidates(pb, perms)["dist"])
    ctx.close()


def test_host_entry_point_in_several_passes(torch_cuda):
    """More than 1 GiB of plans: whp_eval_candidates_host stages them in several passes through one
    buffer (the copy stream waits for the previous pass to be evaluated). 600,000 mid-scale plans
    (1.2 GB of int32 ids): argmin and sampled rows against the oracle, every row against the
    device-resident call."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload("mid")
    pb = wl.problem
    n, n_cand = pb.n_orders, 600_000
    ctx = whp.Context.from_problem(pb)
    perms_dev = torch.empty((n_cand, n), dtype=torch.int32, device="cuda")
    for lo in range(0, n_cand, 100_000):
        perms_dev[lo:lo + 100_000] = W.perms_torch(wl.seed, n, lo, lo + 100_000, "cuda")
    d_dev = torch.zeros(n_cand, dtype=torch.int64, device="cuda")
    o_dev = torch.zeros(n_cand, dtype=torch.float64, device="cuda")
    i_dev = torch.zeros(1, dtype=torch.int64, device="cuda")
    ctx.eval_candidates(perms_dev, dist=d_dev, obj=o_dev)
    ctx.argmin(o_dev, i_dev)
    h = perms_dev.cpu().numpy()
    assert h.nbytes > (1 << 30)
    d, o = np.zeros(n_cand, np.int64), np.zeros(n_cand, np.float64)
    i, v = ctx.eval_candidates_host(h, d, o)
    assert np.array_equal(d, d_dev.cpu().numpy()) and np.array_equal(o, o_dev.cpu().numpy())
    assert i == int(i_dev.item())
    rows = np.unique(np.concatenate([[0, 1, n_cand - 1, 536_870, 536_871],  # around the pass boundary
                                     (W.stream_u64(3, 5, 300) % np.uint64(n_cand)).astype(np.int64)]))
    ref = oracle.eval_candidates(pb, h[rows])
    assert np.array_equal(d[rows], ref["dist"]) and np.array_equal(o[rows], ref["obj"])
    assert np.array_equal(h[rows], W.perm_rows(wl.seed, n, rows))
    one = oracle.eval_candidates(pb, h[i])
    assert one["obj"][0] == v
    # the 16-bit call takes one pass for the same plans (1.2 GB / 2)
    d16, o16 = np.zeros(n_cand, np.int64), np.zeros(n_cand, np.float64)
    i16, v16 = ctx.eval_candidates_host(h.astype(np.uint16), d16, o16)
    assert np.array_equal(d16, d) and np.array_equal(o16, o) and i16 == i and v16 == v
    ctx.close()


def test_routing_and_host_calls_under_cuda_graph_rules(torch_cuda):
    """whp_eval_routing is capturable after one eager call (it allocates nothing); a replay gives
    the oracle's values."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid")
    perms_np = W.perm_rows(2, pb.n_orders, np.arange(200))
    perms = torch.from_numpy(perms_np).cuda()
    ctx = whp.Context.from_problem(pb)
    d = torch.zeros(200, dtype=torch.int64, device="cuda")
    o = torch.zeros(200, dtype=torch.float64, device="cuda")
    ctx.eval_routing(perms, whp.ROUTE_LARGEST_GAP, d, o)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=torch.cuda.Stream()):
        ctx.eval_routing(perms, whp.ROUTE_LARGEST_GAP, d, o)
    d.zero_(), o.zero_()
    g.replay()
    torch.cuda.synchronize()
    ref = oracle.eval_routing(pb, perms_np, oracle.LARGEST_GAP)
    assert np.array_equal(d.cpu().numpy(), ref["dist"]) and np.array_equal(o.cpu().numpy(), ref["obj"])
    del g
    ctx.close()
