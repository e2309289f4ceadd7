"""GPU parity for the routing policies of SURVEY.md §8(f) NEXT-2's second half (readings N5 return,
N6 largest gap): whp_eval_routing against the oracle's orc_eval_routing, bit for bit, on the five
configurations' shapes (stress on a sample of its plans: the oracle needs ~12 ms per stress plan
and policy) and on edge geometries — depot inside and right of the aisles, carts longer than a
warp (shared-memory sort), one-aisle layouts, carts of one pick."""
import os

import numpy as np
import pytest

import oracle
from paper_2110_13693_b200 import workloads as W
from test_gpu_parity import _random_problem

pytestmark = pytest.mark.gpu
CORES = os.cpu_count() or 1


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def gpu_routing(torch, ctx, perms_dev, policy):
    n = perms_dev.shape[0]
    d = torch.full((n,), -1, dtype=torch.int64, device="cuda")
    o = torch.zeros(n, dtype=torch.float64, device="cuda")
    ctx.eval_routing(perms_dev, policy, d, o)
    torch.cuda.synchronize()
    return d.cpu().numpy(), o.cpu().numpy()


def check(torch, ctx, pb, perms, policies=(0, 1, 2), both_kernels=True):
    """Carts of up to 32 picks run the register-resident kernel; `force general` selects the
    shared-memory-list kernel (the only one for larger carts), so both are checked."""
    from paper_2110_13693_b200 import whp
    dev = torch.from_numpy(perms).cuda()
    for pol in policies:
        ref = oracle.eval_routing(pb, perms, pol, threads=CORES)
        for general in ((0, 1) if both_kernels else (0,)):
            ctx.debug_set(whp.DEBUG_FORCE_GENERAL, general)
            d, o = gpu_routing(torch, ctx, dev, pol)
            ctx.debug_set(whp.DEBUG_FORCE_GENERAL, -1)
            bad = np.flatnonzero((d != ref["dist"]) | (o != ref["obj"]))
            assert bad.size == 0, f"policy {pol} general {general}: {bad.size} plans differ, first {bad[:5]}"
            assert np.all(np.abs(o - ref["obj"]) <= 1e-9 * np.abs(ref["obj"]))


@pytest.mark.parametrize("name", ["tiny", "mid"])
def test_routing_every_plan(torch_cuda, name):
    from paper_2110_13693_b200 import whp
    wl = W.make_workload(name)
    pb = wl.problem
    ctx = whp.Context.from_problem(pb)
    check(torch_cuda, ctx, pb, W.perms(wl.seed, pb.n_orders, wl.n_cand))
    ctx.close()


def test_routing_golden_on_gpu(torch_cuda, golden):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    from test_oracle_pins import _golden_problem
    pb = _golden_problem(golden)
    r = golden["routing"]
    perm = np.array([[p for p in golden["plans"] if p["id"] == r["plan"]][0]["perm"]], np.int32)
    ctx = whp.Context.from_problem(pb)
    d, o = gpu_routing(torch, ctx, torch.from_numpy(perm).cuda(), whp.ROUTE_RETURN)
    assert int(d[0]) == r["return_total"] and float(o[0]) == r["return_obj"]
    d, o = gpu_routing(torch, ctx, torch.from_numpy(perm).cuda(), whp.ROUTE_LARGEST_GAP)
    assert int(d[0]) == r["largest_gap_total"] and float(o[0]) == r["largest_gap_obj"]
    ctx.close()


def test_routing_paper_scale_every_plan(torch_cuda):
    """The launch bench.py times: all 16,384 paper-scale plans, both policies, every plan checked."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload("paper")
    pb = wl.problem
    ctx = whp.Context.from_problem(pb)
    perms = W.perms(wl.seed, pb.n_orders, wl.n_cand)
    check(torch, ctx, pb, perms, policies=(1, 2))
    ctx.close()


def test_routing_stress_shape_sampled(torch_cuda):
    """C = 40: the cart's key list no longer fits one key per lane (shared-memory bitonic sort)."""
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    wl = W.make_workload("stress")
    pb = wl.problem
    ctx = whp.Context.from_problem(pb)
    check(torch, ctx, pb, W.perm_rows(wl.seed, pb.n_orders, np.arange(96)), policies=(1, 2))
    ctx.close()


ROUTE_EDGE = [
    dict(NA=1, S=1, K=1, n_skus=1, n_orders=1, qmax=1, C=1),
    dict(NA=1, S=7, K=1, n_skus=5, n_orders=33, qmax=3, C=3),            # one aisle only
    dict(NA=2, S=9, K=3, n_skus=30, n_orders=64, qmax=4, C=9),            # never an inner aisle
    dict(NA=5, S=9, K=3, n_skus=30, n_orders=31, qmax=4, C=4),
    dict(NA=37, S=11, K=33, n_skus=200, n_orders=97, qmax=1, C=1),        # carts of one pick
    dict(NA=64, S=20, K=64, n_skus=500, n_orders=257, qmax=6, C=32, depot=20),  # a full warp of keys
    dict(NA=64, S=20, K=64, n_skus=500, n_orders=257, qmax=6, C=33, depot=63),  # one key too many
    dict(NA=1024, S=30, K=256, n_skus=5000, n_orders=1000, qmax=12, C=40, depot=1023, pitch=3, spacing=7),
    dict(NA=400, S=4095, K=200, n_skus=3000, n_orders=333, qmax=255, C=600),     # limits: q, slots
    dict(NA=8, S=12, K=40, n_skus=100, n_orders=129, qmax=5, C=70),        # many picks per aisle
    dict(NA=5, S=9, K=3, n_skus=30, n_orders=32, qmax=4, C=1000),          # one cart holds all
    dict(NA=12, S=100, K=9, n_skus=1100, n_orders=300, qmax=20, C=1024, depot=6),
    dict(NA=20, S=50, K=9, n_skus=300, n_orders=100, qmax=5, C=20, pitch=1000000, spacing=7),  # 64-bit cart lengths
]


@pytest.mark.parametrize("cfg", ROUTE_EDGE, ids=lambda c: "-".join(f"{k}{v}" for k, v in c.items()))
def test_routing_edge_cases(torch_cuda, cfg):
    from paper_2110_13693_b200 import whp
    pb = _random_problem(23, **cfg)
    ctx = whp.Context.from_problem(pb)
    check(torch_cuda, ctx, pb, W.perm_rows(5, pb.n_orders, np.arange(40)))
    ctx.close()


def test_routing_argument_errors(torch_cuda):
    torch = torch_cuda
    from paper_2110_13693_b200 import whp
    pb = _random_problem(2, NA=5, S=9, K=3, n_skus=30, n_orders=32, qmax=4, C=1025)
    ctx = whp.Context.from_problem(pb)
    perms = torch.from_numpy(W.perm_rows(5, pb.n_orders, np.arange(4))).cuda()
    d = torch.zeros(4, dtype=torch.int64, device="cuda")
    with pytest.raises(whp.WhpError) as e:
        ctx.eval_routing(perms, 3, d)
    assert e.value.status == whp.ERR_INVALID_ARG
    with pytest.raises(whp.WhpError) as e:
        ctx.eval_routing(perms, whp.ROUTE_RETURN, d)
    assert e.value.status == whp.ERR_OUT_OF_RANGE
    ctx.eval_routing(perms, whp.ROUTE_S_SHAPE, d)  # the S-shape path has no such limit
    ctx.eval_routing(perms[:0], whp.ROUTE_RETURN, d)  # empty input: a no-op
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy(), oracle.eval_routing(pb, perms.cpu().numpy(), 0)["dist"])
    ctx.close()
