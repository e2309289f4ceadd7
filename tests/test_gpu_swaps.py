"""GPU parity for the swap-neighbourhood evaluator (a6, D8), the argmin and the trajectory loop
(BASELINE.json configs[4]: "results must match the oracle's trajectory move-for-move")."""
import numpy as np
import pytest

import oracle
from paper_2110_13693_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def gpu_swaps(torch, ctx, base_dev, s, Wn):
    nn = Wn * (Wn - 1) // 2
    d = torch.full((nn,), -1, dtype=torch.int64, device="cuda")
    o = torch.zeros(nn, dtype=torch.float64, device="cuda")
    ctx.eval_swaps(base_dev, s, Wn, d, o)
    torch.cuda.synchronize()
    return d, o


def gpu_trajectory(torch, ctx, base_np, Wn, stride, n_iter):
    """The D8 loop with no host round trip inside an iteration: eval_swaps -> argmin ->
    apply_swap, all on the device; per-iteration results are gathered on the device too."""
    n = len(base_np)
    nn = Wn * (Wn - 1) // 2
    perm = torch.from_numpy(base_np.copy()).cuda()
    d = torch.zeros(nn, dtype=torch.int64, device="cuda")
    o = torch.zeros(nn, dtype=torch.float64, device="cuda")
    idx = torch.zeros(n_iter, dtype=torch.int64, device="cuda")
    val = torch.zeros(n_iter, dtype=torch.float64, device="cuda")
    dist = torch.zeros(n_iter, dtype=torch.int64, device="cuda")
    for it in range(n_iter):
        s = (it * stride) % (n - Wn + 1)
        ctx.eval_swaps(perm, s, Wn, d, o)
        ctx.argmin(o, idx[it:it + 1], val[it:it + 1])
        dist[it:it + 1] = d[idx[it:it + 1]]
        ctx.apply_swap(perm, s, Wn, idx[it:it + 1])
    torch.cuda.synchronize()
    return idx.cpu().numpy(), dist.cpu().numpy(), val.cpu().numpy(), perm.cpu().numpy()


@pytest.mark.parametrize("name,s,Wn", [("tiny", 0, 20), ("tiny", 3, 7), ("mid", 0, 40),
                                       ("mid", 111, 33), ("mid", 467, 33), ("mid", 250, 2)])
def test_swaps_match_oracle_every_neighbour(torch_cuda, name, s, Wn):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem(name)
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(0, pb.n_orders)
    d, o = gpu_swaps(torch, ctx, torch.from_numpy(base).cuda(), s, Wn)
    ref = oracle.eval_swaps(pb, base, s, Wn)
    assert np.array_equal(d.cpu().numpy(), ref["dist"])
    assert np.array_equal(o.cpu().numpy(), ref["obj"])  # bit-identical (canonical sum)
    idx = torch.zeros(1, dtype=torch.int64, device="cuda")
    ctx.argmin(o, idx)
    torch.cuda.synchronize()
    assert int(idx) == oracle.argmin(ref["obj"])
    ctx.close()


def test_swaps_full_length_window(torch_cuda):
    """NEXT-4 groundwork: the window may be the whole plan (all n(n-1)/2 swaps); positions beyond
    the staged region take the global-memory path of the look-up tables."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid", n_orders=300)
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(3, pb.n_orders)
    d, o = gpu_swaps(torch, ctx, torch.from_numpy(base).cuda(), 0, pb.n_orders)
    ref = oracle.eval_swaps(pb, base, 0, pb.n_orders)
    assert np.array_equal(d.cpu().numpy(), ref["dist"])
    assert np.array_equal(o.cpu().numpy(), ref["obj"])
    ctx.close()


@pytest.mark.parametrize("kind", ["swaps", "moves"])
def test_window_longer_than_the_staged_tables(torch_cuda, kind):
    """The neighbour kernels stage 1,024 positions of the prefix / order tables in shared memory;
    a 1,300-wide window reaches past them (global-memory path of the accessors). All 844,350
    swaps (1,688,700 moves) are computed; a sample of them — biased to the far end — is checked
    against the oracle on the materialised plans."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid", n_orders=1300)
    ctx = whp.Context.from_problem(pb)
    n = pb.n_orders
    base = W.base_perm(4, n)
    bd = torch.from_numpy(base).cuda()
    rng = np.random.default_rng(12)
    i = np.concatenate([rng.integers(0, n, 1500), rng.integers(0, 200, 700), rng.integers(1000, n, 800)])
    j = np.concatenate([rng.integers(0, n, 1500), rng.integers(1030, n, 700), rng.integers(1000, n, 800)])
    keep = i != j
    i, j = i[keep], j[keep]
    plans = np.repeat(base[None, :], len(i), axis=0)
    if kind == "swaps":
        i, j = np.minimum(i, j), np.maximum(i, j)
        nn = n * (n - 1) // 2
        idx = i * (2 * n - i - 1) // 2 + (j - i - 1)
        plans[np.arange(len(i)), i], plans[np.arange(len(i)), j] = base[j], base[i]
        d = torch.zeros(nn, dtype=torch.int64, device="cuda")
        o = torch.zeros(nn, dtype=torch.float64, device="cuda")
        ctx.eval_swaps(bd, 0, n, d, o)
    else:
        nn = n * (n - 1)
        idx = i * (n - 1) + np.where(j < i, j, j - 1)
        for r, (a, b) in enumerate(zip(i, j)):
            plans[r] = np.insert(np.delete(base, a), b, base[a])
        d = torch.zeros(nn, dtype=torch.int64, device="cuda")
        o = torch.zeros(nn, dtype=torch.float64, device="cuda")
        ctx.eval_moves(bd, 0, n, d, o)
    torch.cuda.synchronize()
    ref = oracle.eval_candidates(pb, plans)
    sel = torch.from_numpy(idx).cuda()
    assert np.array_equal(d[sel].cpu().numpy(), ref["dist"])
    assert np.array_equal(o[sel].cpu().numpy(), ref["obj"])
    ctx.close()


@pytest.mark.parametrize("margin", ["0", "7", "40"])
def test_swaps_chains_that_leave_the_tabulated_region(torch_cuda, margin):
    """The chain sums cover the window plus a margin; with a tiny margin most chains leave the
    region before they meet the base plan and the neighbour kernel must fall back to scoring
    batch by batch — with the same results."""
    import os
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid")
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(1, pb.n_orders)
    ref = oracle.eval_swaps(pb, base, 60, 36)
    ctx.debug_set(whp.DEBUG_SWAP_MARGIN, int(margin))
    try:
        d, o = gpu_swaps(torch, ctx, torch.from_numpy(base).cuda(), 60, 36)
    finally:
        ctx.debug_set(whp.DEBUG_SWAP_MARGIN, -1)
    assert np.array_equal(d.cpu().numpy(), ref["dist"])
    assert np.array_equal(o.cpu().numpy(), ref["obj"])
    ctx.close()


@pytest.mark.parametrize("n_orders,s,Wn,margin", [(20000, 9000, 28, None), (20000, 9000, 28, "8000"),
                                                  (30000, 21000, 12, None), (30000, 29988, 12, "9000")])
def test_swaps_on_long_plans(torch_cuda, n_orders, s, Wn, margin):
    """Stress-size plans: 20,000 and 30,000 orders are more than the base pass can keep in shared
    memory (12 bytes a position), so its prefix, batch-end and boundary-mark tables are the global
    ones. With a region of 8,000+ positions the hop records (48 bytes a position) do not fit
    shared memory either, so the chain blocks read them from global memory. Swaps and insertion
    moves of a small window against the oracle."""
    import os
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("stress", n_orders=n_orders)
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(2, pb.n_orders)
    ref = oracle.eval_swaps(pb, base, s, Wn)
    ref_m = oracle.eval_moves(pb, base, s, 10)
    if margin is not None:
        ctx.debug_set(whp.DEBUG_SWAP_MARGIN, int(margin))
    try:
        bd = torch.from_numpy(base).cuda()
        d, o = gpu_swaps(torch, ctx, bd, s, Wn)
        md = torch.zeros(90, dtype=torch.int64, device="cuda")
        mo = torch.zeros(90, dtype=torch.float64, device="cuda")
        ctx.eval_moves(bd, s, 10, md, mo)
        torch.cuda.synchronize()
    finally:
        ctx.debug_set(whp.DEBUG_SWAP_MARGIN, -1)
    assert np.array_equal(d.cpu().numpy(), ref["dist"])
    assert np.array_equal(o.cpu().numpy(), ref["obj"])
    assert np.array_equal(md.cpu().numpy(), ref_m["dist"])
    assert np.array_equal(mo.cpu().numpy(), ref_m["obj"])
    ctx.close()


@pytest.mark.parametrize("cfg,s,Wn", [
    # a cart of 9,000 items: the per-segment boundary table of the base pass (segments x C entries)
    # is not built and one thread chases the boundaries
    (dict(NA=30, S=40, K=50, n_skus=800, n_orders=300, qmax=255, C=9000), 100, 24),
    # ~14,000 carts: more than the 8,192 whose class-count prefix (rpre) the base pass builds in
    # shared memory, so the chunk totals go through global memory
    (dict(NA=40, S=50, K=70, n_skus=900, n_orders=20000, qmax=3, C=3), 9000, 12),
    (dict(NA=40, S=50, K=70, n_skus=900, n_orders=20000, qmax=3, C=3), 19988, 12),
])
def test_swaps_beyond_the_shared_memory_tables_of_the_base_pass(torch_cuda, cfg, s, Wn):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    from test_gpu_parity import _random_problem
    pb = _random_problem(21, **cfg)
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(4, pb.n_orders)
    ref = oracle.eval_swaps(pb, base, s, Wn)
    ref_m = oracle.eval_moves(pb, base, s, 8)
    bd = torch.from_numpy(base).cuda()
    d, o = gpu_swaps(torch, ctx, bd, s, Wn)
    md = torch.zeros(56, dtype=torch.int64, device="cuda")
    mo = torch.zeros(56, dtype=torch.float64, device="cuda")
    ctx.eval_moves(bd, s, 8, md, mo)
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy(), ref["dist"])
    assert np.array_equal(o.cpu().numpy(), ref["obj"])
    assert np.array_equal(md.cpu().numpy(), ref_m["dist"])
    assert np.array_equal(mo.cpu().numpy(), ref_m["obj"])
    ctx.close()


def test_swap_stats_count_the_batches_scored_from_their_picks(torch_cuda):
    """One-item orders, C = 5: carts are exactly 5 positions and every boundary stays. A swap
    inside a cart changes nothing (no batch scored); a swap across carts rescores exactly the two
    carts (10 picks). Window of 20 positions = 4 carts: 40 pairs inside a cart, 150 across."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    from test_gpu_parity import _random_problem
    pb = _random_problem(5, NA=12, S=9, K=10, n_skus=80, n_orders=50, qmax=1, C=5)
    ctx = whp.Context.from_problem(pb)
    base = torch.from_numpy(W.base_perm(1, pb.n_orders)).cuda()
    d, o = gpu_swaps(torch, ctx, base, 0, 20)
    assert ctx.get_swap_stats() == (0, 0)          # off by default
    ctx.set_swap_stats(True)
    d2, o2 = gpu_swaps(torch, ctx, base, 0, 20)
    assert ctx.get_swap_stats() == (300, 1500)
    assert torch.equal(d, d2) and torch.equal(o, o2)
    d3, o3 = gpu_swaps(torch, ctx, base, 5, 5)      # one cart: nothing to rescore
    assert ctx.get_swap_stats() == (0, 0)
    ctx.set_swap_stats(False)
    ctx.close()


def test_smaller_opening_order_slips_into_previous_cart(torch_cuda):
    """q = [2,1,3,1], C = 4: swapping positions 2 and 3 (both in the second batch) lets the
    1-item order join the first cart — the incremental evaluator must restart one batch early."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("tiny")
    pb.order_ptr = np.array([0, 2, 3, 6, 7], np.int32)
    pb.item_sku = np.array([0, 11, 22, 33, 5, 17, 39], np.int32)
    pb.cart_capacity = 4
    base = np.arange(4, dtype=np.int32)
    assert oracle.eval_candidates(pb, base, detail=True)["batch_of_pos"][0].tolist() == [0, 0, 1, 1]
    assert oracle.eval_candidates(pb, base[[0, 1, 3, 2]], detail=True)["batch_of_pos"][0].tolist() == [0, 0, 0, 1]
    ctx = whp.Context.from_problem(pb)
    d, o = gpu_swaps(torch, ctx, torch.from_numpy(base).cuda(), 0, 4)
    ref = oracle.eval_swaps(pb, base, 0, 4)
    assert np.array_equal(d.cpu().numpy(), ref["dist"]) and np.array_equal(o.cpu().numpy(), ref["obj"])
    ctx.close()


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_swaps_random_small_problems(torch_cuda, seed):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    from test_gpu_parity import _random_problem
    pb = _random_problem(seed, NA=9, S=6, K=35, n_skus=60, n_orders=70 + seed, qmax=5, C=7 + seed,
                         depot=seed)
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(seed, pb.n_orders)
    for s, Wn in [(0, pb.n_orders), (5, 30)]:
        d, o = gpu_swaps(torch, ctx, torch.from_numpy(base).cuda(), s, Wn)
        ref = oracle.eval_swaps(pb, base, s, Wn)
        assert np.array_equal(d.cpu().numpy(), ref["dist"])
        assert np.array_equal(o.cpu().numpy(), ref["obj"])
    ctx.close()


def test_trajectory_mid_move_for_move(torch_cuda):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid")
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(0, pb.n_orders)
    Wn, stride, n_iter = 32, 16, 40
    ref = oracle.swap_trajectory(pb, base, Wn, stride, n_iter)
    idx, dist, val, perm = gpu_trajectory(torch, ctx, base, Wn, stride, n_iter)
    assert np.array_equal(idx, ref["move"]) and np.array_equal(dist, ref["dist"])
    assert np.array_equal(val, ref["obj"]) and np.array_equal(perm, ref["perm"])
    ctx.close()


def test_trajectory_replayed_from_a_cuda_graph(torch_cuda):
    """After one eager pass (which sizes the context's scratch) every call of the loop is
    asynchronous and allocation-free, so the whole trajectory — and a candidate evaluation with
    its argmin — can be captured in a CUDA graph. A replay must reproduce the oracle's trajectory
    move for move, twice."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid")
    ctx = whp.Context.from_problem(pb)
    n = pb.n_orders
    base_np = W.base_perm(0, n)
    Wn, stride, n_iter = 32, 16, 24
    ref = oracle.swap_trajectory(pb, base_np, Wn, stride, n_iter)
    perms_np = W.perm_rows(5, n, np.arange(300))
    ref_c = oracle.eval_candidates(pb, perms_np)
    nn = Wn * (Wn - 1) // 2
    base0 = torch.from_numpy(base_np.copy()).cuda()
    perm = base0.clone()
    perms = torch.from_numpy(perms_np).cuda()
    d = torch.zeros(nn, dtype=torch.int64, device="cuda")
    o = torch.zeros(nn, dtype=torch.float64, device="cuda")
    idx = torch.zeros(n_iter, dtype=torch.int64, device="cuda")
    val = torch.zeros(n_iter, dtype=torch.float64, device="cuda")
    cd = torch.zeros(300, dtype=torch.int64, device="cuda")
    co = torch.zeros(300, dtype=torch.float64, device="cuda")
    ci = torch.zeros(1, dtype=torch.int64, device="cuda")

    def loop():
        ctx.eval_candidates(perms, dist=cd, obj=co)
        ctx.argmin(co, ci)
        for it in range(n_iter):
            s = (it * stride) % (n - Wn + 1)
            ctx.eval_swaps(perm, s, Wn, d, o)
            ctx.argmin(o, idx[it:it + 1], val[it:it + 1])
            ctx.apply_swap(perm, s, Wn, idx[it:it + 1])

    loop()  # eager: sizes the scratch
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    perm.copy_(base0)
    torch.cuda.synchronize()
    with torch.cuda.graph(g, stream=torch.cuda.Stream()):
        loop()
    for _ in range(2):
        perm.copy_(base0)
        idx.zero_(), val.zero_(), cd.zero_(), co.zero_(), ci.fill_(-1)
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(idx.cpu().numpy(), ref["move"])
        assert np.array_equal(val.cpu().numpy(), ref["obj"])
        assert np.array_equal(perm.cpu().numpy(), ref["perm"])
        assert np.array_equal(cd.cpu().numpy(), ref_c["dist"])
        assert np.array_equal(co.cpu().numpy(), ref_c["obj"])
        assert int(ci.item()) == oracle.argmin(ref_c["obj"])
    del g
    ctx.close()


def test_neighbourhood_config_paper_scale(torch_cuda):
    """configs[4] at full size: W = 256 (32,640 neighbours), stride 128, 100 iterations. The
    oracle re-evaluates every neighbour from scratch (~50 s per iteration), so here: the first
    2 iterations are compared move for move on a window the oracle can afford (full
    neighbourhood, oracle on every neighbour, W = 64), and the full-size run is checked per
    iteration — the applied move's (D, J) equals the oracle's evaluation of the materialised
    permutation, the argmin is the first minimum of the GPU objectives, and sampled neighbours
    equal the oracle."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload("neighbourhood")
    pb = wl.problem
    n = pb.n_orders
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(wl.seed, n)
    # (a) move-for-move against the oracle on a smaller window
    ref = oracle.swap_trajectory(pb, base, 64, 32, 2)
    idx, dist, val, perm = gpu_trajectory(torch, ctx, base, 64, 32, 2)
    assert np.array_equal(idx, ref["move"]) and np.array_equal(val, ref["obj"])
    assert np.array_equal(perm, ref["perm"])
    # (b) the full configuration
    Wn, stride, n_iter = wl.window, wl.stride, wl.n_iter
    idx, dist, val, perm_end = gpu_trajectory(torch, ctx, base, Wn, stride, n_iter)
    perm = base.copy()
    for it in range(n_iter):
        s = (it * stride) % (n - Wn + 1)
        i, j = oracle.decode_neighbour(Wn, int(idx[it]))
        if it % 25 == 0:  # neighbourhood spot check before applying the move
            d, o = gpu_swaps(torch, ctx, torch.from_numpy(perm).cuda(), s, Wn)
            o_np = o.cpu().numpy()
            assert int(idx[it]) == int(np.argmin(o_np))
            for nb in (W.stream_u64(it, 3, 24) % np.uint64(len(o_np))).astype(np.int64):
                a, b = oracle.decode_neighbour(Wn, int(nb))
                p = perm.copy()
                p[s + a], p[s + b] = p[s + b], p[s + a]
                one = oracle.eval_candidates(pb, p)
                assert one["obj"][0] == o_np[nb] and one["dist"][0] == int(d[nb])
        perm[s + i], perm[s + j] = perm[s + j], perm[s + i]
        one = oracle.eval_candidates(pb, perm)
        assert one["dist"][0] == dist[it] and one["obj"][0] == val[it]
    assert np.array_equal(perm, perm_end)
    ctx.close()


# ---- NEXT-1: NHATC outer loop on the device ---------------------------------------------------
@pytest.mark.parametrize("name,n_cand,n_outer,beta", [("tiny", 64, 6, 1.5), ("mid", 512, 5, 1.25)])
def test_nhatc_solve_matches_oracle_loop(torch_cuda, name, n_cand, n_outer, beta):
    """eval -> argmin -> update, n_outer times with no host round trip: winners, their D and J and
    the final multipliers equal the oracle's loop bit for bit (rounding order fixed by reading N1)."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem(name)
    perms = W.perms(0, pb.n_orders, n_cand)
    ctx = whp.Context.from_problem(pb)
    idx = torch.zeros(n_outer, dtype=torch.int64, device="cuda")
    dist = torch.zeros(n_outer, dtype=torch.int64, device="cuda")
    obj = torch.zeros(n_outer, dtype=torch.float64, device="cuda")
    ctx.nhatc_solve(torch.from_numpy(perms).cuda(), n_outer, beta, idx, dist, obj)
    torch.cuda.synchronize()
    ref = oracle.nhatc_loop(pb, perms, n_outer, beta)
    assert np.array_equal(idx.cpu().numpy(), ref["idx"])
    assert np.array_equal(dist.cpu().numpy(), ref["dist"])
    assert np.array_equal(obj.cpu().numpy(), ref["obj"])
    t, v, w = ctx.get_penalty()
    assert np.array_equal(t, pb.t) and np.array_equal(v, ref["v"]) and np.array_equal(w, ref["w"])
    ctx.close()


def test_nhatc_update_single_step(torch_cuda, ):
    torch = torch_cuda
    import json, os
    from paper_2110_13693_b200 import whp
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "worked_examples.json")))["nhatc_update"]
    pb = W.make_problem("tiny")
    ctx = whp.Context.from_problem(pb)
    ctx.set_penalty(g["t"], g["v"], g["w"])
    rows = torch.tensor([[9, 9, 9, 9], g["r"]], dtype=torch.int32, device="cuda")
    ctx.nhatc_update(rows, torch.tensor([1], dtype=torch.int64, device="cuda"), g["beta"])
    t, v, w = ctx.get_penalty()
    assert v.tolist() == g["v_new"] and w.tolist() == g["w_new"] and t.tolist() == g["t"]
    ctx.close()


# ---- NEXT-4: insertion moves ----------------------------------------------------------------------
def gpu_moves(torch, ctx, base_dev, s, Wn):
    nn = Wn * (Wn - 1)
    d = torch.full((nn,), -1, dtype=torch.int64, device="cuda")
    o = torch.zeros(nn, dtype=torch.float64, device="cuda")
    ctx.eval_moves(base_dev, s, Wn, d, o)
    torch.cuda.synchronize()
    return d, o


@pytest.mark.parametrize("name,s,Wn", [("tiny", 0, 20), ("tiny", 3, 7), ("mid", 0, 30),
                                       ("mid", 111, 25), ("mid", 470, 30), ("mid", 250, 2)])
def test_moves_match_oracle_every_neighbour(torch_cuda, name, s, Wn):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem(name)
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(0, pb.n_orders)
    d, o = gpu_moves(torch, ctx, torch.from_numpy(base).cuda(), s, Wn)
    ref = oracle.eval_moves(pb, base, s, Wn)
    assert np.array_equal(d.cpu().numpy(), ref["dist"])
    assert np.array_equal(o.cpu().numpy(), ref["obj"])
    ctx.close()


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_moves_random_small_problems_and_trajectory(torch_cuda, seed):
    """Small random problems (many slips and resynchronisations), then a short descent:
    eval_moves -> argmin -> apply_move on the device against the same loop with the oracle."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    rng = np.random.default_rng(seed)
    n = 48
    q = rng.integers(1, 5, size=n)
    ptr = np.concatenate([[0], np.cumsum(q)]).astype(np.int32)
    pb = W.Problem(n_aisles=9, slots_per_side=6, slot_pitch=1, aisle_spacing=2, depot_aisle=seed,
                   sku_loc=rng.integers(0, 108, size=30).astype(np.int32),
                   sku_class=rng.integers(0, 5, size=30).astype(np.int32), n_classes=5,
                   order_ptr=ptr, item_sku=rng.integers(0, 30, size=int(ptr[-1])).astype(np.int32),
                   cart_capacity=6, t=rng.uniform(0, 9, 5), v=rng.uniform(0, 1, 5), w=rng.uniform(0, 1, 5))
    ctx = whp.Context.from_problem(pb)
    perm = W.base_perm(seed, n).copy()
    dev = torch.from_numpy(perm).cuda()
    idx = torch.zeros(1, dtype=torch.int64, device="cuda")
    for it in range(4):
        s0, Wn = (it * 7) % (n - 16 + 1), 16
        d, o = gpu_moves(torch, ctx, dev, s0, Wn)
        ref = oracle.eval_moves(pb, perm, s0, Wn)
        assert np.array_equal(d.cpu().numpy(), ref["dist"]) and np.array_equal(o.cpu().numpy(), ref["obj"])
        ctx.argmin(o, idx)
        ctx.apply_move(dev, s0, Wn, idx)
        torch.cuda.synchronize()
        k = oracle.argmin(ref["obj"])
        assert int(idx) == k
        i, jr = divmod(k, Wn - 1)
        j = jr if jr < i else jr + 1
        moved = perm[s0 + i]
        perm = np.insert(np.delete(perm, s0 + i), s0 + j, moved).astype(np.int32)
        assert np.array_equal(dev.cpu().numpy(), perm)
    ctx.close()


@pytest.mark.parametrize("margin", ["0", "9"])
def test_moves_chains_that_leave_the_tabulated_region(torch_cuda, margin):
    import os
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid")
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(4, pb.n_orders)
    ref = oracle.eval_moves(pb, base, 200, 24)
    ctx.debug_set(whp.DEBUG_SWAP_MARGIN, int(margin))
    try:
        d, o = gpu_moves(torch, ctx, torch.from_numpy(base).cuda(), 200, 24)
    finally:
        ctx.debug_set(whp.DEBUG_SWAP_MARGIN, -1)
    assert np.array_equal(d.cpu().numpy(), ref["dist"]) and np.array_equal(o.cpu().numpy(), ref["obj"])
    ctx.close()


def test_moves_paper_scale_sampled(torch_cuda):
    """All 65,280 moves of a 256-wide window at paper scale; the oracle re-evaluates sampled ones."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload("paper")
    pb = wl.problem
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(wl.seed, pb.n_orders)
    s0, Wn = 1280, 256
    d, o = gpu_moves(torch, ctx, torch.from_numpy(base).cuda(), s0, Wn)
    d, o = d.cpu().numpy(), o.cpu().numpy()
    rows = np.unique((W.stream_u64(5, 3, 150) % np.uint64(Wn * (Wn - 1))).astype(np.int64))
    for k in rows:
        i, jr = divmod(int(k), Wn - 1)
        j = jr if jr < i else jr + 1
        seq = np.insert(np.delete(base, s0 + i), s0 + j, base[s0 + i]).astype(np.int32)
        one = oracle.eval_candidates(pb, seq)
        assert d[k] == one["dist"][0] and o[k] == one["obj"][0]
    ctx.close()


def test_two_contexts_on_two_streams_as_bench_issues_a_step(torch_cuda):
    """bench.py's step (--overlap 1): candidate evaluation + argmin on one stream, neighbourhood
    pass + argmin + apply on a second stream with a context of its own ("one context per
    stream", include/whp.h), forked and joined by events every step. Both halves must still
    equal the oracle: all candidates bit for bit, the trajectory move for move."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid")
    n = pb.n_orders
    ctx, ctx_nb = whp.Context.from_problem(pb), whp.Context.from_problem(pb)
    n_cand, Wn, stride, n_iter = 1024, 32, 16, 24
    rows = W.perm_rows(3, n, np.arange(n_cand))
    perms = torch.from_numpy(rows).cuda()
    base = W.base_perm(5, n)
    ref = oracle.eval_candidates(pb, rows)
    ref_tr = oracle.swap_trajectory(pb, base, Wn, stride, n_iter)

    nn = Wn * (Wn - 1) // 2
    perm = torch.from_numpy(base.copy()).cuda()
    dist = torch.zeros(n_cand, dtype=torch.int64, device="cuda")
    pen = torch.zeros(n_cand, dtype=torch.float64, device="cuda")
    obj = torch.zeros(n_cand, dtype=torch.float64, device="cuda")
    nbat = torch.zeros(n_cand, dtype=torch.int32, device="cuda")
    bhash = torch.zeros(n_cand, dtype=torch.int64, device="cuda")
    best = torch.zeros(n_iter, dtype=torch.int64, device="cuda")
    sd = torch.zeros(nn, dtype=torch.int64, device="cuda")
    so = torch.zeros(nn, dtype=torch.float64, device="cuda")
    move = torch.zeros(n_iter, dtype=torch.int64, device="cuda")
    mval = torch.zeros(n_iter, dtype=torch.float64, device="cuda")
    main, side = torch.cuda.current_stream(), torch.cuda.Stream(priority=-1)
    fork_ev, join_ev = torch.cuda.Event(), torch.cuda.Event()
    torch.cuda.synchronize()
    for it in range(n_iter):
        s = (it * stride) % (n - Wn + 1)
        fork_ev.record(main)
        side.wait_event(fork_ev)
        with torch.cuda.stream(side):
            ctx_nb.eval_swaps(perm, s, Wn, sd, so)
            ctx_nb.argmin(so, move[it:it + 1], mval[it:it + 1])
            ctx_nb.apply_swap(perm, s, Wn, move[it:it + 1])
            join_ev.record(side)
        dist.fill_(-1)
        ctx.eval_candidates(perms, dist=dist, penalty=pen, obj=obj, n_batches=nbat,
                            batch_hash=bhash)
        ctx.argmin(obj, best[it:it + 1])
        main.wait_event(join_ev)
    torch.cuda.synchronize()
    assert np.array_equal(dist.cpu().numpy(), ref["dist"])
    assert np.array_equal(obj.cpu().numpy(), ref["obj"])
    assert np.array_equal(pen.cpu().numpy(), ref["penalty"])
    assert np.array_equal(nbat.cpu().numpy(), ref["n_batches"])
    assert np.array_equal(bhash.cpu().numpy().view(np.uint64), ref["batch_hash"])
    assert np.all(best.cpu().numpy() == oracle.argmin(ref["obj"]))
    assert np.array_equal(move.cpu().numpy(), ref_tr["move"])
    assert np.array_equal(mval.cpu().numpy(), ref_tr["obj"])
    assert np.array_equal(perm.cpu().numpy(), ref_tr["perm"])
    ctx.close()
    ctx_nb.close()


def test_neighbour_index_decode_at_row_boundaries_of_a_4000_wide_window(torch_cuda):
    """The neighbour kernel turns n into (i', j') by a float square-root estimate made exact by
    integer correction loops (32-bit below 32,768 positions). At W = 4,000 — the whole
    paper-scale plan, 7,998,000 swaps — (2W-1)^2 no longer fits a float mantissa, so the estimate
    is off near the row boundaries: the first and last neighbour of many rows, and random ones,
    against the oracle on the materialised plans."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("paper")
    ctx = whp.Context.from_problem(pb)
    n = pb.n_orders
    base = W.base_perm(6, n)
    rng = np.random.default_rng(21)
    rows = np.unique(np.concatenate([np.arange(0, 6), np.arange(n - 8, n - 1), [1000, 2047, 2048, 2896, 3000],
                                     rng.integers(0, n - 1, 60)]))
    i = np.concatenate([rows, rows, rng.integers(0, n - 1, 150)])
    j = np.concatenate([rows + 1, np.full(len(rows), n - 1), np.zeros(150, dtype=np.int64)])
    j[2 * len(rows):] = rng.integers(i[2 * len(rows):] + 1, n)
    idx = i * (2 * n - i - 1) // 2 + (j - i - 1)
    plans = np.repeat(base[None, :], len(i), axis=0)
    plans[np.arange(len(i)), i], plans[np.arange(len(i)), j] = base[j], base[i]
    nn = n * (n - 1) // 2
    d = torch.zeros(nn, dtype=torch.int64, device="cuda")
    o = torch.zeros(nn, dtype=torch.float64, device="cuda")
    ctx.eval_swaps(torch.from_numpy(base).cuda(), 0, n, d, o)
    torch.cuda.synchronize()
    ref = oracle.eval_candidates(pb, plans)
    sel = torch.from_numpy(idx).cuda()
    assert np.array_equal(d[sel].cpu().numpy(), ref["dist"])
    assert np.array_equal(o[sel].cpu().numpy(), ref["obj"])
    ctx.close()


def test_nhatc_solve_replayed_from_a_cuda_graph(torch_cuda):
    """"the loop captured in a CUDA graph". After one eager call (which
    sizes the response scratch) whp_nhatc_solve neither allocates nor synchronises, so the whole
    outer loop — walk, argmin, record, multiplier update, n_outer times — is captured once and
    replayed; every replay restarts from the same multipliers and must reproduce the oracle's
    loop (reading N1) bit for bit."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("mid")
    n_cand, n_outer, beta = 384, 4, 1.25
    perms_np = W.perms(3, pb.n_orders, n_cand)
    ref = oracle.nhatc_loop(pb, perms_np, n_outer, beta)
    ctx = whp.Context.from_problem(pb)
    perms = torch.from_numpy(perms_np).cuda()
    idx = torch.zeros(n_outer, dtype=torch.int64, device="cuda")
    dist = torch.zeros(n_outer, dtype=torch.int64, device="cuda")
    obj = torch.zeros(n_outer, dtype=torch.float64, device="cuda")
    ctx.nhatc_solve(perms, n_outer, beta, idx, dist, obj)  # eager: sizes the scratch
    torch.cuda.synchronize()
    ctx.set_penalty(pb.t, pb.v, pb.w)
    # the multipliers live in the context: a device-side snapshot restores them before a replay
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=torch.cuda.Stream()):
        ctx.nhatc_solve(perms, n_outer, beta, idx, dist, obj)
    for _ in range(2):
        ctx.set_penalty(pb.t, pb.v, pb.w)
        idx.fill_(-1), dist.zero_(), obj.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(idx.cpu().numpy(), ref["idx"])
        assert np.array_equal(dist.cpu().numpy(), ref["dist"])
        assert np.array_equal(obj.cpu().numpy(), ref["obj"])
        t, v, w = ctx.get_penalty()
        assert np.array_equal(v, ref["v"]) and np.array_equal(w, ref["w"])
    del g
    ctx.close()


def test_apply_swap_ignores_indices_that_are_no_neighbour(torch_cuda):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("tiny")
    ctx = whp.Context.from_problem(pb)
    base = W.base_perm(0, pb.n_orders)
    Wn, s = 6, 9
    for bad in (-1, -3, -(1 << 40), Wn * (Wn - 1) // 2, 1 << 40):
        perm = torch.from_numpy(base.copy()).cuda()
        ctx.apply_swap(perm, s, Wn, torch.tensor([bad], dtype=torch.int64, device="cuda"))
        ctx.apply_move(perm, s, Wn, torch.tensor([bad if bad < 0 else max(bad, Wn * (Wn - 1))],
                                                 dtype=torch.int64, device="cuda"))
        torch.cuda.synchronize()
        assert np.array_equal(perm.cpu().numpy(), base), bad
    perm = torch.from_numpy(base.copy()).cuda()
    last = Wn * (Wn - 1) // 2 - 1  # (i', j') = (W-2, W-1)
    ctx.apply_swap(perm, s, Wn, torch.tensor([last], dtype=torch.int64, device="cuda"))
    torch.cuda.synchronize()
    want = base.copy()
    want[s + Wn - 2], want[s + Wn - 1] = want[s + Wn - 1], want[s + Wn - 2]
    assert np.array_equal(perm.cpu().numpy(), want)
    ctx.close()


def test_binding_rejects_short_or_foreign_buffers(torch_cuda):
    """The C side cannot see a tensor's size: the binding checks it before the call."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = W.make_problem("tiny")
    ctx = whp.Context.from_problem(pb)
    perms = torch.from_numpy(W.perms(0, pb.n_orders, 8)).cuda()
    with pytest.raises(ValueError):
        ctx.eval_candidates(perms, dist=torch.zeros(7, dtype=torch.int64, device="cuda"))
    with pytest.raises(ValueError):
        ctx.eval_candidates(perms, resp=torch.zeros(8 * pb.n_classes - 1, dtype=torch.int32, device="cuda"))
    with pytest.raises(ValueError):
        ctx.eval_swaps(perms[0], 0, 6, obj=torch.zeros(14, dtype=torch.float64, device="cuda"))
    with pytest.raises(ValueError):
        ctx.eval_moves(perms[0], 0, 6, obj=torch.zeros(29, dtype=torch.float64, device="cuda"))
    with pytest.raises(ValueError):
        ctx.argmin(torch.zeros(4, dtype=torch.float64, device="cuda"), torch.zeros(1, dtype=torch.int32, device="cuda"))
    with pytest.raises(ValueError):  # int64 host plans would be misread as int32
        ctx.eval_candidates_host(W.perms(0, pb.n_orders, 8).astype(np.int64))
    with pytest.raises(ValueError):
        ctx.eval_candidates_host(W.perms(0, pb.n_orders, 8), dist=np.zeros(7, np.int64))
    with pytest.raises(whp.WhpError):
        ctx.debug_set(99, 1)
    h = np.ascontiguousarray(W.perms(0, pb.n_orders, 8))
    d, o = np.zeros(8, np.int64), np.zeros(8, np.float64)
    i, v = ctx.eval_candidates_host(h, d, o)
    ref = oracle.eval_candidates(pb, h)
    assert np.array_equal(d, ref["dist"]) and np.array_equal(o, ref["obj"]) and i == oracle.argmin(ref["obj"])
    ctx.close()
