"""Pins for the oracle (CPU only): closed forms, invariants, brute force, hand-worked examples.

Each test cites the definition (DESIGN.md §2 / SURVEY.md §8(c)) it pins. Nothing here touches
the CUDA path. The helpers below are deliberately written in a different style from
oracle/whp_oracle.c (python sets, itertools, exact rationals) so that a shared mistake is
unlikely.
"""
import itertools
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2110_13693_b200 import workloads as W

TINY = (4, 10, 1, 3, 0)  # NA, S, pitch, spacing, depot (BASELINE.json configs[1])


# ---------- independent helpers (tests only) -------------------------------------------------
def _point(geom, loc):
    NA, S, p, P, a0 = geom
    return loc // (2 * S), (loc % S + 1) * p


def _walk(geom, u, v):
    """D0 metric written from the layout picture: same aisle -> along it; else out through the
    nearer cross-aisle (front y=0, back y=A), across, and in."""
    NA, S, p, P, a0 = geom
    A = (S + 1) * p
    (a1, y1), (a2, y2) = u, v
    if a1 == a2:
        return abs(y1 - y2)
    return abs(a1 - a2) * P + min(y1 + y2, (A - y1) + (A - y2))


def _brute_route(geom, locs):
    pts = sorted({_point(geom, l) for l in locs})
    depot = (geom[4], 0)
    best = None
    for order in itertools.permutations(pts):
        tour = [depot, *order, depot]
        d = sum(_walk(geom, tour[i], tour[i + 1]) for i in range(len(tour) - 1))
        best = d if best is None or d < best else best
    return best


def _py_plan(pb, perm):
    """D1-D5 with python sets; returns (batch_of_pos, per-batch loc lists, r)."""
    q = np.diff(pb.order_ptr)
    bop, b, load = [], 0, 0
    for o in perm:
        if load > 0 and load + q[o] > pb.cart_capacity:
            b, load = b + 1, 0
        bop.append(b)
        load += q[o]
    batches = [[] for _ in range(b + 1)]
    classes = [set() for _ in range(b + 1)]
    for pos, o in enumerate(perm):
        for it in range(pb.order_ptr[o], pb.order_ptr[o + 1]):
            sku = pb.item_sku[it]
            batches[bop[pos]].append(int(pb.sku_loc[sku]))
            classes[bop[pos]].add(int(pb.sku_class[sku]))
    r = [sum(1 for cs in classes if k in cs) for k in range(pb.n_classes)]
    return bop, batches, r


def _exact_penalty(r, t, v, w):
    """phi as an exact rational (fp64 inputs are rationals), then rounded once."""
    tot = Fraction(0)
    for rk, tk, vk, wk in zip(r, t, v, w):
        c = Fraction(float(tk)) - int(rk)
        tot += Fraction(float(vk)) * c + (Fraction(float(wk)) * c) ** 2
    return tot


def _golden_problem(golden):
    g, pp = golden["geometry"], golden["plan_problem"]
    ptr = np.cumsum([0] + [len(o) for o in pp["orders"]])
    return W.Problem(
        n_aisles=g["n_aisles"], slots_per_side=g["slots_per_side"], slot_pitch=g["slot_pitch"],
        aisle_spacing=g["aisle_spacing"], depot_aisle=g["depot_aisle"],
        sku_loc=np.array(pp["sku_loc"], np.int32), sku_class=np.array(pp["sku_class"], np.int32),
        n_classes=pp["n_classes"], order_ptr=ptr.astype(np.int32),
        item_sku=np.array([s for o in pp["orders"] for s in o], np.int32),
        cart_capacity=pp["cart_capacity"], t=np.array(pp["t"]), v=np.array(pp["v"]),
        w=np.array(pp["w"]))


# ---------- E1-E6: hand-worked examples -------------------------------------------------------
def test_golden_batches(golden):
    geom = tuple(golden["geometry"][k] for k in
                 ("n_aisles", "slots_per_side", "slot_pitch", "aisle_spacing", "depot_aisle"))
    for ex in golden["batches"]:
        assert oracle.batch_distance(geom, ex["locs"]) == ex["dist"], ex["id"]
        assert oracle.optimal_route(geom, ex["locs"]) == ex["optimal"], ex["id"]
        assert _brute_route(geom, ex["locs"]) == ex["optimal"], ex["id"]


def test_golden_plans(golden):
    pb = _golden_problem(golden)
    perms = np.array([p["perm"] for p in golden["plans"]], np.int32)
    out = oracle.eval_candidates(pb, perms, detail=True)
    for i, ex in enumerate(golden["plans"]):
        assert out["batch_of_pos"][i].tolist() == ex["batch_of_pos"], ex["id"]
        assert int(out["dist"][i]) == ex["dist"], ex["id"]
        assert out["resp"][i].tolist() == ex["resp"], ex["id"]
        assert out["penalty"][i] == ex["penalty"], ex["id"]  # dyadic data: exact in any order
        assert out["obj"][i] == ex["obj"], ex["id"]
        assert int(out["batch_hash"][i]) == ex["batch_hash"], ex["id"]
        assert int(out["n_batches"][i]) == len(ex["batch_dist"]), ex["id"]
        bd, _ = oracle.eval_candidate_batches(pb, perms[i])
        assert bd.tolist() == ex["batch_dist"], ex["id"]
        if "n_distinct" in ex:
            assert int(out["n_distinct"][i]) == ex["n_distinct"]
        if "batch_optimal" in ex:
            _, batches, _ = _py_plan(pb, perms[i])
            geom = (pb.n_aisles, pb.slots_per_side, pb.slot_pitch, pb.aisle_spacing,
                    pb.depot_aisle)
            assert [oracle.optimal_route(geom, b) for b in batches] == ex["batch_optimal"]
    assert oracle.argmin(out["obj"][:2]) == golden["argmin_E4_E5"]


def test_golden_swap_E6(golden):
    pb = _golden_problem(golden)
    e4, e6 = golden["plans"][0], golden["plans"][2]
    s, Wn = e6["window"]
    sw = oracle.eval_swaps(pb, np.array(e4["perm"], np.int32), s, Wn)
    n = e6["neighbour_index"]
    assert oracle.decode_neighbour(Wn, n) == tuple(e6["pair"])
    assert int(sw["dist"][n]) == e6["dist"] and sw["obj"][n] == e6["obj"]


# ---------- P1/P2: closed forms of D4 (north_star) ---------------------------------------------
@pytest.mark.parametrize("geom", [TINY, (20, 50, 1, 3, 0), (7, 13, 2, 5, 0)])
def test_single_aisle_closed_form(geom):
    NA, S, p, P, a0 = geom
    for loc in range(2 * NA * S):
        a, depth = loc // (2 * S), (loc % S + 1) * p
        assert oracle.batch_distance(geom, [loc]) == 2 * a * P + 2 * depth
        # one aisle, several picks: out to the deepest and back — also the true optimum
        other = (loc // S) * S + (loc * 7 + 3) % S
        deepest = max(depth, (other % S + 1) * p)
        assert oracle.batch_distance(geom, [loc, other, loc]) == 2 * a * P + 2 * deepest
        if loc % 17 == 0:
            assert oracle.optimal_route(geom, [loc, other]) == 2 * a * P + 2 * deepest


def test_even_aisles_full_traversals_only():
    geom = (20, 50, 1, 3, 0)
    NA, S, p, P, a0 = geom
    A = (S + 1) * p
    rng = np.random.default_rng(1)
    for _ in range(300):
        m = int(rng.choice([2, 4, 6, 8]))
        aisles = rng.choice(NA, size=m, replace=False)
        locs = []
        for a in aisles:
            for _ in range(int(rng.integers(1, 4))):
                locs.append(int(a) * 2 * S + int(rng.integers(0, 2 * S)))
        d = oracle.batch_distance(geom, locs)
        assert d == 2 * int(aisles.max()) * P + m * A  # independent of every depth
        # adding a pick in a visited aisle that is not the last one never changes it
        not_last = int(np.sort(aisles)[0])
        assert oracle.batch_distance(geom, locs + [not_last * 2 * S + 3]) == d


def test_odd_aisles_last_aisle_return():
    geom = (20, 50, 1, 3, 0)
    NA, S, p, P, a0 = geom
    A = (S + 1) * p
    rng = np.random.default_rng(2)
    for _ in range(300):
        m = int(rng.choice([1, 3, 5, 7]))
        aisles = np.sort(rng.choice(NA, size=m, replace=False))
        locs, deepest_last = [], 0
        for a in aisles:
            for _ in range(int(rng.integers(1, 4))):
                slot = int(rng.integers(0, S))
                locs.append(int(a) * 2 * S + int(rng.integers(0, 2)) * S + slot)
                if a == aisles[-1]:
                    deepest_last = max(deepest_last, (slot + 1) * p)
        assert oracle.batch_distance(geom, locs) == (2 * int(aisles[-1]) * P + (m - 1) * A
                                                     + 2 * deepest_last)


def test_nonzero_depot_horizontal_term():
    # D4's H for a depot in the middle: out to the leftmost, across, back from the rightmost
    geom = (9, 6, 1, 4, 4)
    S, P, A = 6, 4, 7
    locs = [2 * 2 * S + 1, 7 * 2 * S + 2]  # aisles 2 and 7, m = 2
    assert oracle.batch_distance(geom, locs) == P * ((4 - 2) + (7 - 2) + (7 - 4)) + 2 * A
    locs = [6 * 2 * S + 1]  # single aisle right of the depot, depth 2
    assert oracle.batch_distance(geom, locs) == P * (2 + 0 + 2) + 2 * 2


# ---------- P3: S-shape >= exhaustive optimum; metric cross-checked --------------------------
def test_sshape_not_below_optimal_on_every_tiny_batch():
    wl = W.make_workload("tiny")
    pb = wl.problem
    perms = W.perms(wl.seed, pb.n_orders, wl.n_cand)
    n_checked = 0
    for c in range(wl.n_cand):
        bd, _ = oracle.eval_candidate_batches(pb, perms[c])
        _, batches, _ = _py_plan(pb, perms[c])
        assert len(bd) == len(batches)
        for d, locs in zip(bd, batches):
            opt = oracle.optimal_route(TINY, locs)
            assert opt >= 0 and d >= opt  # cart capacity 8 => at most 8 distinct locations
            n_checked += 1
            if c < 4:  # the C enumeration against the itertools one
                assert opt == _brute_route(TINY, locs)
    assert n_checked > 400


def test_optimal_route_matches_itertools_on_random_sets():
    rng = np.random.default_rng(3)
    geom = (6, 8, 2, 5, 0)
    for _ in range(60):
        locs = rng.integers(0, 2 * 6 * 8, size=int(rng.integers(1, 7))).tolist()
        assert oracle.optimal_route(geom, locs) == _brute_route(geom, locs)
        assert oracle.batch_distance(geom, locs) >= _brute_route(geom, locs)


# ---------- P4: invariances of dist_b ---------------------------------------------------------
def test_batch_distance_invariances():
    rng = np.random.default_rng(4)
    geom = (20, 50, 1, 3, 0)
    S = 50
    for _ in range(200):
        locs = rng.integers(0, 2000, size=int(rng.integers(1, 25)))
        d = oracle.batch_distance(geom, locs)
        assert oracle.batch_distance(geom, rng.permutation(locs)) == d
        assert oracle.batch_distance(geom, np.concatenate([locs, locs[:3]])) == d
        flipped = (locs // (2 * S)) * 2 * S + (1 - (locs % (2 * S)) // S) * S + locs % S
        assert oracle.batch_distance(geom, flipped) == d


# ---------- P5: batching invariants -------------------------------------------------------------
@pytest.mark.parametrize("name", ["tiny", "mid"])
def test_batching_invariants(name):
    wl = W.make_workload(name)
    pb = wl.problem
    n = min(wl.n_cand, 48)
    perms = W.perm_rows(wl.seed, pb.n_orders, np.arange(n))
    out = oracle.eval_candidates(pb, perms, detail=True)
    q = np.diff(pb.order_ptr)
    C = pb.cart_capacity
    for c in range(n):
        bop = out["batch_of_pos"][c]
        assert bop[0] == 0 and np.all(np.diff(bop) >= 0) and np.all(np.diff(bop) <= 1)
        nb = int(out["n_batches"][c])
        assert nb == bop[-1] + 1 and nb >= -(-pb.n_items // C)
        loads = np.bincount(bop, weights=q[perms[c]], minlength=nb).astype(int)
        assert loads.max() <= C and loads.min() >= 1
        starts = np.flatnonzero(np.diff(bop, prepend=-1))
        for b in range(nb - 1):  # greedy: the next order did not fit
            assert loads[b] + q[perms[c][starts[b + 1]]] > C
        assert int(out["batch_hash"][c]) == sum((int(s) + 1) * (2 * b + 1)
                                                for b, s in enumerate(starts)) % (1 << 64)
        # P8: responses recounted with sets; per-candidate python restatement
        pbop, batches, r = _py_plan(pb, perms[c])
        assert pbop == bop.tolist() and r == out["resp"][c].tolist()
        assert max(r) <= nb and sum(r) >= nb
        assert int(out["n_distinct"][c]) == sum(len(set(b)) for b in batches)
        assert int(out["dist"][c]) == sum(oracle.batch_distance(pb, b) for b in batches)


def test_one_big_cart_is_permutation_invariant():
    pb = W.make_problem("tiny")
    pb.cart_capacity = pb.n_items
    perms = W.perm_rows(0, pb.n_orders, np.arange(16))
    out = oracle.eval_candidates(pb, perms)
    assert np.all(out["n_batches"] == 1) and len(set(out["dist"].tolist())) == 1
    all_locs = pb.sku_loc[pb.item_sku]
    assert int(out["dist"][0]) == oracle.batch_distance(pb, all_locs)


def test_every_order_fills_the_cart():
    pb = W.make_problem("tiny")
    q = 3
    n_orders = 12
    pb.order_ptr = (np.arange(n_orders + 1) * q).astype(np.int32)
    pb.item_sku = (W.stream_u64(5, 77, n_orders * q) % np.uint64(pb.n_skus)).astype(np.int32)
    pb.cart_capacity = q
    perms = W.perm_rows(1, n_orders, np.arange(8))
    out = oracle.eval_candidates(pb, perms)
    per_order = sum(oracle.batch_distance(pb, pb.sku_loc[pb.item_sku[o * q:(o + 1) * q]])
                    for o in range(n_orders))
    assert np.all(out["n_batches"] == n_orders) and np.all(out["dist"] == per_order)


# ---------- P6: penalty ---------------------------------------------------------------------------
def test_penalty_closed_forms():
    assert oracle.penalty([3], [5.0], [0.5], [0.25]) == 0.5 * 2.0 + (0.25 * 2.0) ** 2  # K = 1
    r = np.arange(40, dtype=np.int32)
    assert oracle.penalty(r, r.astype(float), np.ones(40), np.ones(40)) == 0.0  # t = r
    assert oracle.penalty(r, r + 1.0, np.zeros(40), np.zeros(40)) == 0.0  # v = w = 0
    # sign of c = t - r: a response above target with v > 0, w = 0 gives a NEGATIVE linear term
    assert oracle.penalty([4], [1.0], [2.0], [0.0]) == -6.0
    assert oracle.penalty([4], [1.0], [0.0], [2.0]) == 36.0  # (w c)^2, not w c^2


@pytest.mark.parametrize("K", [1, 4, 20, 31, 32, 33, 200, 256])
def test_penalty_against_exact_rational(K):
    rng = np.random.default_rng(K)
    for scale in ("unit", "log"):
        r = rng.integers(0, 400, size=K).astype(np.int32)
        t = rng.uniform(0, 400, size=K)
        v = rng.uniform(0, 1, size=K) if scale == "unit" else 10 ** rng.uniform(-3, 3, K)
        w = rng.uniform(0, 1, size=K) if scale == "unit" else 10 ** rng.uniform(-3, 3, K)
        exact = _exact_penalty(r, t, v, w)
        mag = sum(abs(float(vk * (tk - rk))) + float(wk * (tk - rk)) ** 2
                  for rk, tk, vk, wk in zip(r, t, v, w))
        assert abs(Fraction(oracle.penalty(r, t, v, w)) - exact) <= Fraction(1e-12) * Fraction(mag)


def test_objective_is_distance_plus_penalty():
    wl = W.make_workload("mid")
    pb = wl.problem
    perms = W.perm_rows(0, pb.n_orders, np.arange(8))
    out = oracle.eval_candidates(pb, perms, detail=True)
    for c in range(8):
        assert out["penalty"][c] == oracle.penalty(out["resp"][c], pb.t, pb.v, pb.w)
        assert out["obj"][c] == float(out["dist"][c]) + out["penalty"][c]
    pb.v = np.zeros_like(pb.v)
    pb.w = np.zeros_like(pb.w)
    out0 = oracle.eval_candidates(pb, perms)
    assert np.all(out0["obj"] == out0["dist"].astype(float))


# ---------- P7: swap neighbourhood ------------------------------------------------------------------
def test_swaps_equal_materialised_permutations():
    wl = W.make_workload("mid")
    pb = wl.problem
    base = W.base_perm(0, pb.n_orders)
    s, Wn = 37, 12
    sw = oracle.eval_swaps(pb, base, s, Wn)
    base_out = oracle.eval_candidates(pb, base, detail=True)
    q = np.diff(pb.order_ptr)
    n = 0
    for i in range(Wn):
        for j in range(i + 1, Wn):
            assert oracle.decode_neighbour(Wn, n) == (i, j)
            assert n == i * (2 * Wn - i - 1) // 2 + (j - i - 1)
            p = base.copy()
            p[s + i], p[s + j] = p[s + j], p[s + i]
            one = oracle.eval_candidates(pb, p)
            assert sw["dist"][n] == one["dist"][0] and sw["obj"][n] == one["obj"][0]
            bop = base_out["batch_of_pos"][0]
            first_of_batch = s + i == 0 or bop[s + i - 1] != bop[s + i]
            if bop[s + i] == bop[s + j] and not first_of_batch:
                # both orders inside one batch, and the batch's opening order unchanged (a
                # smaller opening order could slip into the previous cart): nothing changes
                assert sw["obj"][n] == base_out["obj"][0]
            if q[base[s + i]] == q[base[s + j]]:
                assert one["n_batches"][0] == base_out["n_batches"][0]
            n += 1


def test_trajectory_applies_argmin_each_iteration():
    pb = W.make_problem("tiny")
    base = W.base_perm(0, pb.n_orders)
    tr = oracle.swap_trajectory(pb, base, 6, 3, 5)
    perm = base.copy()
    for it in range(5):
        s = (it * 3) % (pb.n_orders - 6 + 1)
        sw = oracle.eval_swaps(pb, perm, s, 6)
        best = int(np.argmin(sw["obj"]))  # numpy: first minimum
        assert tr["move"][it] == best and tr["obj"][it] == sw["obj"][best]
        i, j = oracle.decode_neighbour(6, best)
        perm[s + i], perm[s + j] = perm[s + j], perm[s + i]
    assert perm.tolist() == tr["perm"].tolist()


# ---------- P9: argmin ----------------------------------------------------------------------------------
def test_argmin_first_minimum():
    assert oracle.argmin(np.full(17, 3.25)) == 0
    x = np.array([5.0, 2.0, 7.0, 2.0, 2.0, 9.0])
    assert oracle.argmin(x) == 1
    rng = np.random.default_rng(9)
    for _ in range(50):
        x = rng.integers(0, 6, size=int(rng.integers(1, 40))).astype(float)
        assert oracle.argmin(x) == int(np.argmin(x))


# ---- NEXT-1: NHATC multiplier update (reading N1) -------------------------------------------
def test_nhatc_update_golden(golden):
    g = golden["nhatc_update"]
    v, w = oracle.nhatc_update(g["r"], g["t"], g["v"], g["w"], g["beta"])
    assert v.tolist() == g["v_new"] and w.tolist() == g["w_new"]


def test_nhatc_update_special_cases_and_exact_rational():
    from fractions import Fraction
    rng = np.random.default_rng(3)
    K = 37
    r = rng.integers(0, 50, K)
    t, v, w = rng.uniform(0, 40, K), rng.uniform(-3, 3, K), rng.uniform(0, 2, K)
    v0, w0 = oracle.nhatc_update(r, t, v, np.zeros(K), 3.0)
    assert np.array_equal(v0, v) and not w0.any()                  # w = 0: multipliers stay
    v1, w1 = oracle.nhatc_update(r, r.astype(np.float64), v, w, 1.0)
    assert np.array_equal(v1, v) and np.array_equal(w1, w)         # consistent plan, beta = 1
    v2, w2 = oracle.nhatc_update(r, t, v, w, 2.5)
    assert np.array_equal(w2, 2.5 * w)
    for k in range(K):                                             # v' = v + 2 w^2 (t - r), exactly
        c = Fraction(float(t[k])) - int(r[k])
        exact = Fraction(float(v[k])) + 2 * Fraction(float(w[k])) ** 2 * c
        bound = 4 * 2.0 ** -53 * (abs(v[k]) + 2 * w[k] ** 2 * abs(float(c)))
        assert abs(float(Fraction(float(v2[k])) - exact)) <= bound
    # the multiplier term moves against the inconsistency: (v' - v).c = 2 sum (w c)^2 >= 0
    c = t - r
    assert np.dot(v2 - v, c) >= 0.0


def test_nhatc_loop_is_eval_argmin_update():
    pb = W.make_problem("tiny")
    perms = W.perms(0, pb.n_orders, 16)
    h = oracle.nhatc_loop(pb, perms, 3, 1.5)
    import copy
    q = copy.copy(pb)
    for it in range(3):
        out = oracle.eval_candidates(q, perms, detail=True)
        i = int(np.argmin(out["obj"]))
        assert h["idx"][it] == i and h["obj"][it] == out["obj"][i] and h["dist"][it] == out["dist"][i]
        q.v, q.w = oracle.nhatc_update(out["resp"][i], q.t, q.v, q.w, 1.5)
    assert np.array_equal(h["v"], q.v) and np.array_equal(h["w"], q.w)
    assert np.array_equal(h["w"], pb.w * 1.5 * 1.5 * 1.5)


# ---- NEXT-2: leg sums (reading N2) ----------------------------------------------------------------
def test_legsum_golden(golden):
    geom = tuple(golden["geometry"][k] for k in
                 ("n_aisles", "slots_per_side", "slot_pitch", "aisle_spacing", "depot_aisle"))
    for tour in golden["legsum"]["tours"]:
        assert oracle.tour_length(geom, tour["locs"]) == tour["len"] == sum(tour["legs"])
    pb = _golden_problem(golden)
    plan = next(p for p in golden["plans"] if p["id"] == golden["legsum"]["plan"])
    assert oracle.eval_legsum(pb, np.array(plan["perm"]))[0] == golden["legsum"]["total"]


def test_tour_closed_forms_and_optimal_route_is_the_best_ordering():
    import itertools
    geom = (5, 9, 2, 3, 1)  # aisles, slots/side, pitch, spacing, depot aisle
    S2 = 2 * 9
    # one pick: out and back = the single-aisle closed form of D4 (m = 1)
    for loc in (0, 7, 25, 44, 89):
        a, depth = loc // S2, (loc % 9 + 1) * 2
        assert oracle.tour_length(geom, [loc]) == 2 * (abs(a - 1) * 3 + depth) == oracle.batch_distance(geom, [loc])
    # a repeated location adds nothing; a tour and its reverse are equally long
    assert oracle.tour_length(geom, [7, 7, 30]) == oracle.tour_length(geom, [7, 30])
    rng = np.random.default_rng(4)
    for _ in range(30):
        locs = rng.integers(0, 5 * S2, size=rng.integers(1, 7)).tolist()
        assert oracle.tour_length(geom, locs) == oracle.tour_length(geom, locs[::-1])
        # the exhaustive optimum (P3's routine) is the minimum of the tour length over orderings
        best = min(oracle.tour_length(geom, list(p)) for p in itertools.permutations(locs))
        assert best == oracle.optimal_route(geom, locs) <= oracle.tour_length(geom, locs)


def test_legsum_is_the_sum_of_cart_tours():
    pb = W.make_problem("tiny")
    perms = W.perms(0, pb.n_orders, 8)
    got = oracle.eval_legsum(pb, perms)
    ref = oracle.eval_candidates(pb, perms, detail=True)
    for c in range(8):
        total = 0
        bop = ref["batch_of_pos"][c]
        for b in range(ref["n_batches"][c]):
            locs = [int(pb.sku_loc[s]) for pos in np.nonzero(bop == b)[0]
                    for s in pb.item_sku[pb.order_ptr[perms[c, pos]]:pb.order_ptr[perms[c, pos] + 1]]]
            total += oracle.tour_length(pb, locs)
        assert got[c] == total


# ---- NEXT-3: K-means slotting (reading N3) ---------------------------------------------------------
def test_kmeans_hand_worked():
    """Frequencies [5,1,1,6,1,5], k=2: lo=1, hi=6, step 2.5: c = [2.25, 4.75]; SKUs 0,3,5 -> cluster 1
    (|5-4.75| = .25, |6-4.75| = 1.25), SKUs 1,2,4 -> cluster 0; centroids 1 and 16/3 (stable).
    Cluster 1 ranks first: order 0,3,5,1,2,4 over the locations of aisle 0 (S=2, depot aisle 0):
    i -> slot i div 2, side i mod 2 -> loc = side*2 + slot: 0,2,1,3; then aisle 1: 4,6."""
    items = [0] * 5 + [1] + [2] + [3] * 6 + [4] + [5] * 5
    out = oracle.kmeans_slotting((3, 2, 1, 3, 0), 6, items, 2, 1, 3)
    assert out["freq"].tolist() == [5, 1, 1, 6, 1, 5]
    assert out["assign"].tolist() == [1, 0, 0, 1, 0, 1]
    assert out["centroids"].tolist() == [1.0, 16.0 / 3.0]
    assert out["sku_loc"].tolist() == [0, 3, 4, 2, 6, 1]
    assert out["sku_class"].tolist() == [1, 0, 0, 1, 0, 1]


def test_kmeans_invariants():
    from fractions import Fraction
    pb = W.make_problem("mid")
    k, Z = 10, 2
    prev_sse = None
    for iters in range(0, 6):
        out = oracle.kmeans_slotting(pb, pb.n_skus, pb.item_sku, k, Z, iters)
        f, a, c = out["freq"], out["assign"], out["centroids"]
        assert f.sum() == pb.n_items and np.array_equal(f, np.bincount(pb.item_sku, minlength=pb.n_skus))
        # nearest centroid, ties to the lowest index
        d = np.abs(f[:, None].astype(np.float64) - c[None, :])
        assert np.array_equal(a, np.argmin(d, axis=1))
        # Lloyd's iterations never increase the within-cluster sum of squares
        sse = float(((f - c[a]) ** 2).sum())
        assert prev_sse is None or sse <= prev_sse * (1 + 1e-12)
        prev_sse = sse
    # slotting: injective, clusters contiguous in the location order, frequent clusters first
    loc = out["sku_loc"]
    assert len(set(loc.tolist())) == pb.n_skus
    S2 = 2 * pb.slots_per_side
    order_index = (loc // S2) * S2 + (loc % pb.slots_per_side) * 2 + (loc % S2) // pb.slots_per_side
    by_pos = np.argsort(order_index)
    cl = a[by_pos]
    change = np.nonzero(np.diff(cl))[0]
    assert len(change) == len(np.unique(a)) - 1                   # every cluster is one run
    cents = c[cl[np.concatenate([[0], change + 1])]]
    assert np.all(np.diff(cents) <= 0)                             # largest centroid first
    zone = (loc % pb.slots_per_side) * Z // pb.slots_per_side
    assert np.array_equal(out["sku_class"], a * Z + zone)
    # with iters >= 1 a centroid of a non-empty cluster is the exact mean of its members at the
    # last update: check on the converged state (assignment stable between iters 5 and 6)
    out6 = oracle.kmeans_slotting(pb, pb.n_skus, pb.item_sku, k, Z, 60)
    out7 = oracle.kmeans_slotting(pb, pb.n_skus, pb.item_sku, k, Z, 61)
    assert np.array_equal(out6["assign"], out7["assign"])
    for j in np.unique(out7["assign"]):
        m = out7["freq"][out7["assign"] == j]
        assert Fraction(float(out7["centroids"][j])) == Fraction(float(int(m.sum()) / len(m)))


# ---- NEXT-4: insertion moves (reading N4) ------------------------------------------------------------
def test_moves_equal_materialised_sequences_and_adjacent_moves_are_swaps(golden):
    pb = W.make_problem("tiny")
    base = W.base_perm(2, pb.n_orders)
    s, Wn = 3, 9
    mv = oracle.eval_moves(pb, base, s, Wn)
    sw = oracle.eval_swaps(pb, base, s, Wn)
    n = 0
    for i in range(Wn):
        for j in range(Wn):
            if i == j:
                continue
            seq = np.delete(base, s + i)                      # built with numpy, not by the oracle
            seq = np.insert(seq, s + j, base[s + i])
            one = oracle.eval_candidates(pb, seq.astype(np.int32))
            assert mv["dist"][n] == one["dist"][0] and mv["obj"][n] == one["obj"][0]
            assert n == i * (Wn - 1) + (j if j < i else j - 1)
            if abs(i - j) == 1:                               # an adjacent move is a swap
                a, b = min(i, j), max(i, j)
                k = a * (2 * Wn - a - 1) // 2 + (b - a - 1)
                assert mv["dist"][n] == sw["dist"][k] and mv["obj"][n] == sw["obj"][k]
            n += 1
    # E4 -> E6 of the hand-worked examples: moving position 1 to position 2 is the swap (1, 2)
    gp = _golden_problem(golden)
    e6 = next(p for p in golden["plans"] if p["id"] == "E6")
    m = oracle.eval_moves(gp, np.arange(6, dtype=np.int32), 0, 6)
    assert m["dist"][1 * 5 + 1] == e6["dist"] and m["obj"][1 * 5 + 1] == e6["obj"]


# ---------- host wrappers and memory safety of the checker itself --------------------------------
def test_threaded_wrappers_equal_the_single_thread_routines():
    """`threads=` only spreads plans / neighbourhood rows over host threads (full-size GPU parity
    tests use it); every value must be the one the single-threaded call gives."""
    pb = W.make_problem("mid")
    base = W.base_perm(0, pb.n_orders)
    for s, Wn in ((11, 2), (11, 3), (0, 7), (460, 40), (5, 41)):
        a = oracle.eval_swaps(pb, base, s, Wn)
        b = oracle.eval_swaps(pb, base, s, Wn, threads=4)
        assert np.array_equal(a["dist"], b["dist"]) and np.array_equal(a["obj"], b["obj"])
    perms = W.perms(0, pb.n_orders, 333)
    a = oracle.eval_candidates(pb, perms, detail=True)
    b = oracle.eval_candidates(pb, perms, detail=True, threads=5)
    for k in a:
        assert np.array_equal(a[k], b[k]), k


def test_oracle_runs_clean_under_address_and_undefined_sanitizers(tmp_path):
    """the oracle under -fsanitize=address,undefined. A separate process (the
    sanitizer runtime must be preloaded) drives every exported routine on tiny / mid inputs; any
    report aborts it."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    so = str(tmp_path / "libwhp_oracle_san.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-std=c99", "-ffp-contract=off", "-fsanitize=address,undefined",
                           "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-shared", "-fPIC",
                           "-o", so, os.path.join(root, "oracle", "whp_oracle.c")])
    asan = subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()
    script = f"""
import sys
sys.path.insert(0, {root!r})
import numpy as np
import oracle.binding as B
B.build = lambda force=False: {so!r}
import oracle
from paper_2110_13693_b200 import workloads as W
for name, n_cand, s, Wn in (("tiny", 64, 3, 9), ("mid", 96, 450, 24)):
    pb = W.make_problem(name)
    perms = W.perms(0, pb.n_orders, n_cand)
    out = oracle.eval_candidates(pb, perms, detail=True, threads=2)
    oracle.argmin(out["obj"])
    oracle.eval_candidate_batches(pb, perms[0])
    oracle.eval_swaps(pb, perms[1], s, Wn, threads=2)
    oracle.eval_moves(pb, perms[2], s, min(Wn, 12))
    oracle.swap_trajectory(pb, perms[3], min(Wn, 10), 5, 3)
    oracle.eval_legsum(pb, perms[:8])
    oracle.nhatc_loop(pb, perms[:16], 2, 1.5)
    for pol in (0, 1, 2):
        oracle.eval_routing(pb, perms[:8], pol, threads=2)
    oracle.kmeans_slotting(pb, pb.n_skus, pb.item_sku, 3, 1, 4)
pb = W.make_problem("tiny")
oracle.optimal_route(pb, pb.sku_loc[:8])
oracle.batch_distance(pb, pb.sku_loc[:5])
oracle.tour_length(pb, pb.sku_loc[:6])
oracle.batch_return_distance(pb, pb.sku_loc[:9])
oracle.batch_largest_gap_distance(pb, pb.sku_loc[:9])
print("SANITIZED_OK")
"""
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    r = subprocess.run([sys.executable, "-c", script], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "SANITIZED_OK" in r.stdout, r.stderr[-3000:]


# ---------- NEXT-2, second half: return and largest-gap routing (readings N5, N6) ------------------
def _aisle_table(geom, locs):
    """{aisle: sorted distinct depths} — the per-aisle depth table, with python sets."""
    tab = {}
    for l in locs:
        a, y = _point(geom, l)
        tab.setdefault(a, set()).add(y)
    return {a: sorted(ys) for a, ys in tab.items()}


def _tour_len_and_cover(geom, way, locs):
    """Length of the closed walk through the waypoints under the independent D0 metric, and
    whether every pick lies on one of its in-aisle segments."""
    total = sum(_walk(geom, way[i], way[i + 1]) for i in range(len(way) - 1))
    covered = set()
    for (a1, y1), (a2, y2) in zip(way[:-1], way[1:]):
        if a1 == a2:
            for l in locs:
                a, y = _point(geom, l)
                if a == a1 and min(y1, y2) <= y <= max(y1, y2):
                    covered.add(l)
    return total, covered == set(locs)


def _return_tour(geom, locs):
    NA, S, p, P, a0 = geom
    tab = _aisle_table(geom, locs)
    way = [(a0, 0)]
    # depot -> leftmost visited aisle -> sweep to the rightmost -> depot, all along the front
    for a in sorted(tab):
        way += [(a, 0), (a, tab[a][-1]), (a, 0)]
    way.append((a0, 0))
    return way


def _largest_gap_tour(geom, locs):
    NA, S, p, P, a0 = geom
    A = (S + 1) * p
    tab = _aisle_table(geom, locs)
    aisles = sorted(tab)
    if len(aisles) == 1:
        a = aisles[0]
        return [(a0, 0), (a, 0), (a, tab[a][-1]), (a, 0), (a0, 0)]
    first, last, mid = aisles[0], aisles[-1], aisles[1:-1]
    cut = {}
    for a in mid:  # (front reach, back reach) around the largest gap; ties -> first
        ys = [0] + tab[a] + [A]
        k = max(range(len(ys) - 1), key=lambda i: (ys[i + 1] - ys[i], -i))
        cut[a] = (ys[k], ys[k + 1])
    def front_entry(a):
        return [(a, 0), (a, cut[a][0]), (a, 0)] if cut[a][0] > 0 else []
    way = [(a0, 0)]
    for a in reversed([x for x in mid if x <= a0]):  # on the way out along the front cross-aisle
        way += front_entry(a)
    way += [(first, 0), (first, A)]
    for a in mid:  # along the back cross-aisle
        if cut[a][1] < A:
            way += [(a, A), (a, cut[a][1]), (a, A)]
    way += [(last, A), (last, 0)]
    for a in reversed([x for x in mid if x > a0]):  # home along the front cross-aisle
        way += front_entry(a)
    way.append((a0, 0))
    return way


def test_routing_golden(golden):
    geom = TINY
    r = golden["routing"]
    for ex in r["batches"]:
        assert oracle.batch_return_distance(geom, ex["locs"]) == ex["return"], ex["id"]
        assert oracle.batch_largest_gap_distance(geom, ex["locs"]) == ex["largest_gap"], ex["id"]
    pb = _golden_problem(golden)
    perm = np.array([p for p in golden["plans"] if p["id"] == r["plan"]][0]["perm"], np.int32)
    ret = oracle.eval_routing(pb, perm, oracle.RETURN)
    lg = oracle.eval_routing(pb, perm, oracle.LARGEST_GAP)
    assert int(ret["dist"][0]) == r["return_total"] and float(ret["obj"][0]) == r["return_obj"]
    assert int(lg["dist"][0]) == r["largest_gap_total"] and float(lg["obj"][0]) == r["largest_gap_obj"]


@pytest.mark.parametrize("geom", [TINY, (7, 9, 2, 5, 3), (20, 50, 1, 3, 0), (12, 30, 3, 4, 11)])
def test_routing_equals_explicit_tours_that_visit_every_pick(geom):
    """N5 / N6 are lengths of real walks: build each tour waypoint by waypoint, check that every
    pick lies on it, and add its legs with the test's own D0 metric."""
    NA, S, p, P, a0 = geom
    rng = np.random.default_rng(hash(geom) % (1 << 31))
    for trial in range(150):
        n = int(rng.integers(1, 13))
        locs = rng.integers(0, 2 * NA * S, n).tolist()
        if trial % 5 == 0:  # few aisles, many picks per aisle
            aisles = rng.integers(0, NA, 2)
            locs = [int(a) * 2 * S + int(x) for a, x in zip(rng.choice(aisles, n), rng.integers(0, 2 * S, n))]
        for tour, fn in ((_return_tour, oracle.batch_return_distance),
                         (_largest_gap_tour, oracle.batch_largest_gap_distance)):
            length, covered = _tour_len_and_cover(geom, tour(geom, locs), locs)
            assert covered, (geom, locs, tour.__name__)
            assert fn(geom, locs) == length, (geom, locs, tour.__name__)


def test_routing_closed_forms_bounds_and_invariances():
    rng = np.random.default_rng(5)
    for geom in (TINY, (6, 8, 2, 5, 2)):
        NA, S, p, P, a0 = geom
        A = (S + 1) * p
        for loc in range(2 * NA * S):  # one pick: the m = 1 closed form of north_star (P1)
            a, y = _point(geom, loc)
            assert oracle.batch_return_distance(geom, [loc]) == 2 * abs(a - a0) * P + 2 * y
            assert oracle.batch_largest_gap_distance(geom, [loc]) == 2 * abs(a - a0) * P + 2 * y
        for _ in range(200):
            locs = rng.integers(0, 2 * NA * S, int(rng.integers(1, 8))).tolist()
            ret, lg = oracle.batch_return_distance(geom, locs), oracle.batch_largest_gap_distance(geom, locs)
            opt = _brute_route(geom, locs)
            assert ret >= opt and lg >= opt  # both are tours: never below the exhaustive optimum
            # invariant to order, repeats and the side of the aisle (P4)
            shuffled = list(rng.permutation(locs + locs[:2]))
            flipped = [l + S if (l % (2 * S)) < S else l - S for l in locs]
            for other in (shuffled, flipped):
                assert oracle.batch_return_distance(geom, other) == ret
                assert oracle.batch_largest_gap_distance(geom, other) == lg
            # the table the policies read: return = H + 2 * sum of the per-aisle maxima
            tab = _aisle_table(geom, locs)
            H = P * (abs(a0 - min(tab)) + (max(tab) - min(tab)) + abs(max(tab) - a0))
            assert ret == H + 2 * sum(ys[-1] for ys in tab.values())
            # largest gap of an aisle = the best way to reach all its picks by one walk in from
            # the front and one in from the back: brute force over where the two walks stop
            if len(tab) >= 3:
                want = H + 2 * A
                for a in sorted(tab)[1:-1]:
                    ys = tab[a]
                    want += min(2 * f + 2 * (A - b) for f, b in zip([0] + ys, ys + [A]))
                assert lg == want


def test_routing_evaluator_shares_batching_and_penalty_with_the_s_shape_path():
    """Policy 0 of eval_routing is D4: it must reproduce eval_candidates (which pins the new
    function's batching, responses and penalty); the other policies differ only in the cart
    lengths, recomputed here per cart from python-side batching."""
    for name in ("tiny", "mid"):
        pb = W.make_problem(name)
        perms = W.perms(1, pb.n_orders, 24)
        ref = oracle.eval_candidates(pb, perms)
        s0 = oracle.eval_routing(pb, perms, oracle.S_SHAPE, threads=3)
        assert np.array_equal(s0["dist"], ref["dist"]) and np.array_equal(s0["obj"], ref["obj"])
        for pol, fn in ((oracle.RETURN, oracle.batch_return_distance),
                        (oracle.LARGEST_GAP, oracle.batch_largest_gap_distance)):
            out = oracle.eval_routing(pb, perms, pol)
            for c in range(6):
                bop, batches, r = _py_plan(pb, perms[c])
                D = sum(fn(pb, b) for b in batches)
                assert out["dist"][c] == D
                assert out["obj"][c] == float(D) + ref["penalty"][c]
    with pytest.raises(ValueError):
        oracle.eval_routing(W.make_problem("tiny"), W.perms(1, 20, 2), 3)
