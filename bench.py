#!/usr/bin/env python
"""bench.py — one JSON line for the candidate picking-plan evaluation path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--overlap 0|1]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

A step is one pass of the whole hot path (SURVEY.md §8(a) rows a1–a7) on the paper-scale
workload (BASELINE.json configs[2] + configs[3], "paper" / "neighbourhood" in workloads.py):
    whp_eval_candidates on 16,384 candidate plans (a1–a5)  -> whp_argmin (a7)
    whp_eval_swaps on the 32,640-neighbour window of the trajectory plan (a6) -> whp_argmin
    -> whp_apply_swap (the trajectory of configs[3] advances one iteration per step).
The two lines are independent of each other; with --overlap 1 (default) they run on two streams,
one context each, forked and joined by events inside every step.
`value` = candidate plans per second over the whole step, inputs resident in HBM. Multi-GPU:
candidates are independent, so each rank evaluates its own 16,384 plans (weak scaling), no
data-path collective; time = max over ranks. `--impl reference` times the oracle (oracle/, a
plain single-threaded CPU program) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2110_13693_b200 import harness, workloads as W  # noqa: E402

WORKLOAD = "paper"  # BASELINE.json configs[2] (the third listed): the config the metric is quoted on
CPU_SAMPLE = 8192   # candidates the oracle is timed on for cpu_baseline (~12 s on one core)
REF_SAMPLE = 256    # candidates per step of --impl reference: 1/64 of the 16,384 of a step
REF_WINDOW = 32     # and the 496 swaps of a 32-wide window: ~1/66 of the step's 32,640 neighbours
LEGS = ("step", "sustained", "e2e", "next", "stress", "cpu")  # --legs; "step" is the contract line
SUSTAIN_S = 2.5     # the `sustained` leg repeats the step for at least this long
KERNEL_PASS = 32    # steps of the separate pass that times the candidate evaluation by events


def config_dict(pb, n_cand, world, wl_nb):
    return {"workload": "paper-scale (BASELINE.json configs[3rd]): 400 aisles x 250 slots/side, "
                        "100k SKUs, Zipf(1.0), K=200",
            "n_orders": pb.n_orders, "n_items": pb.n_items, "cart_capacity": pb.cart_capacity,
            "candidates_per_gpu": n_cand, "global_candidates": n_cand * world,
            "neighbourhood": {"window": wl_nb.window, "stride": wl_nb.stride,
                              "neighbours": wl_nb.window * (wl_nb.window - 1) // 2},
            "parallelism": f"candidates sharded x{world}, tables replicated, no collective",
            "l2": "permutation input 262 MB per step > 126 MB L2 (no flush needed)"}


def run_reference(args):
    """The oracle as it stands, single thread, on the box's host cores; rank 0 only."""
    rank, _, world = harness.dist_env()
    if rank != 0:
        return 0
    import oracle
    wl = W.make_workload(WORKLOAD)
    pb = wl.problem
    wl_nb = W.make_workload("neighbourhood")
    n = REF_SAMPLE
    perms = W.perm_rows(wl.seed, pb.n_orders, np.arange(n))
    base = np.ascontiguousarray(perms[0])
    n_nb = REF_WINDOW * (REF_WINDOW - 1) // 2

    def step():  # the same rows as a step of our arm (a1-a7), on a 1/64 sample of its units
        out = oracle.eval_candidates(pb, perms)
        best = oracle.argmin(out["obj"])
        sw = oracle.eval_swaps(pb, base, 0, REF_WINDOW)
        return best, oracle.argmin(sw["obj"])
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    line = {
        "impl": "reference", "metric": "candidate_plans_per_s", "value": value,
        "unit": "candidate plans/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int64+f64", "data": "synthetic",
        "picks_per_s": value * pb.n_items,
        "config": config_dict(pb, wl.n_cand, 1, wl_nb),
        "cpu_baseline": {"value": value, "unit": "candidate plans/s", "cores": 1,
                         "kind": "oracle",
                         "sample": f"per step: {n} of the 16,384 paper-scale candidates (a1-a5 + "
                                   f"argmin) and the {n_nb} swaps of a {REF_WINDOW}-wide window out "
                                   "of the 32,640 of a step (a6 + argmin), every neighbour "
                                   "re-evaluated from scratch"},
        "e2e": {"value": value, "unit": "candidate plans/s", "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def stress_leg(torch, whp, dev, local_rank, peaks, counters):
    """BASELINE.json configs[5] at its full 65,536 plans: one launch
    of whp_eval_candidates over 5.24 GB of plans generated in HBM, timed by CUDA events."""
    import oracle
    wls = W.make_workload("stress")
    pbs = wls.problem
    ns, ncs = pbs.n_orders, wls.n_cand
    ctx_s = whp.Context.from_problem(pbs, device=local_rank)
    sperms = torch.empty((ncs, ns), dtype=torch.int32, device=dev)
    for lo_s in range(0, ncs, 4096):
        sperms[lo_s:lo_s + 4096] = W.perms_torch(wls.seed, ns, lo_s, lo_s + 4096, dev)
    sd = torch.zeros(ncs, dtype=torch.int64, device=dev)
    so = torch.zeros(ncs, dtype=torch.float64, device=dev)
    sh = torch.zeros(ncs, dtype=torch.int64, device=dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(3):
        ctx_s.eval_candidates(sperms, dist=sd, obj=so, batch_hash=sh)
    torch.cuda.synchronize()
    reps = 10
    ev0.record()
    for _ in range(reps):
        ctx_s.eval_candidates(sperms, dist=sd, obj=so, batch_hash=sh)
    ev1.record()
    torch.cuda.synchronize()
    st_ms = ev0.elapsed_time(ev1) / reps
    sb = harness.algorithmic_bytes_per_candidate(ns, pbs.n_items)
    st_ach = sb["survey"] * ncs / (st_ms * 1e-3) / 1e9
    # spot check against the oracle (all 65,536 plans are compared in tests/test_gpu_fullsize.py)
    rows_s = np.array([0, 1, 4097, ncs - 1])
    ref_s = oracle.eval_candidates(pbs, sperms[torch.from_numpy(rows_s).to(dev)].cpu().numpy())
    stress = {"workload": "stress (BASELINE.json configs[5th]): 20,000 orders, "
                          f"{pbs.n_items} items, C=40, K=32, Zipf(1.2), {ncs} plans in one launch",
              "ms": st_ms, "value": ncs / (st_ms * 1e-3), "unit": "candidate plans/s",
              "picks_per_s": ncs * pbs.n_items / (st_ms * 1e-3),
              "bytes_per_candidate": sb["survey"], "achieved": st_ach, "peak": peaks["hbm_gbs"],
              "unit_achieved": "GB/s", "frac": st_ach / peaks["hbm_gbs"],
              "frac_hbm_compulsory": sb["hbm_compulsory"] * ncs / (st_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
              "traffic": counters.get("stress", {}).get("dram_bytes"),
              "reps": reps, "input_bytes": int(sperms.numel() * 4),
              "sampled_rows_equal_oracle": bool(
                  np.array_equal(ref_s["obj"], so.cpu().numpy()[rows_s])
                  and np.array_equal(ref_s["dist"], sd.cpu().numpy()[rows_s]))}
    ctx_s.close()
    del sperms, sd, so, sh
    torch.cuda.empty_cache()
    return stress


def run_ours(args):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback "
                           "(use --impl reference for the oracle arm)")
    from paper_2110_13693_b200 import whp
    rank, local_rank, world = harness.init_dist("nccl")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    legs = set(LEGS) if args.legs == "all" else set(args.legs.split(","))
    if not legs <= set(LEGS):
        raise SystemExit(f"--legs takes a comma list of {LEGS}")
    if not args.sustain:
        legs.discard("sustained")
    if not args.stress:
        legs.discard("stress")
    if "step" not in legs:  # profiling runs: only the stress launch (no JSON contract line)
        if rank == 0 and "stress" in legs:
            print(json.dumps({"impl": "ours", "legs": sorted(legs),
                              "stress": stress_leg(torch, whp, dev, local_rank,
                                                   harness.measured_peaks(ROOT),
                                                   harness.ncu_counters(ROOT))}))
        return 0

    wl = W.make_workload(WORKLOAD)
    wl_nb = W.make_workload("neighbourhood")
    pb = wl.problem
    n, n_cand = pb.n_orders, wl.n_cand
    ctx = whp.Context.from_problem(pb, device=local_rank)
    if args.k1_warps:
        ctx.debug_set(4, args.k1_warps)  # WHP_DEBUG_K1_WARPS
    lo, hi = harness.weak_rows(n_cand, rank)
    perms = W.perms_torch(wl.seed, n, lo, hi, dev)  # resident in HBM before the clock starts
    dist = torch.zeros(n_cand, dtype=torch.int64, device=dev)
    pen = torch.zeros(n_cand, dtype=torch.float64, device=dev)
    obj = torch.zeros(n_cand, dtype=torch.float64, device=dev)
    nbat = torch.zeros(n_cand, dtype=torch.int32, device=dev)
    bhash = torch.zeros(n_cand, dtype=torch.int64, device=dev)
    idx = torch.zeros(1, dtype=torch.int64, device=dev)
    val = torch.zeros(1, dtype=torch.float64, device=dev)
    Wn, stride = wl_nb.window, wl_nb.stride
    nn = Wn * (Wn - 1) // 2
    base = torch.from_numpy(W.base_perm(wl.seed + rank, n)).to(dev)
    sdist = torch.zeros(nn, dtype=torch.int64, device=dev)
    sobj = torch.zeros(nn, dtype=torch.float64, device=dev)
    sidx = torch.zeros(1, dtype=torch.int64, device=dev)
    # Host buffers of the e2e leg are filled now: for a second or two after a large host-side
    # copy / conversion the H2D copies that follow it run ~20 % slower (measured: 3.2 ms instead
    # of 2.6 ms per 131 MB call), so the buffers must be at rest long before they are timed.
    h_perms = h16 = None
    if "e2e" in legs:
        h_perms = torch.empty((n_cand, n), dtype=torch.int32).pin_memory()
        h_perms.copy_(perms)
        h16 = torch.from_numpy(perms.cpu().numpy().astype(np.uint16).view(np.int16)).pin_memory()
    it_counter = [0]
    # The candidate evaluation's own duration (roofline.kernel_ms) comes from a separate pass
    # AFTER the timed region (KERNEL_PASS more steps of the same two-stream step, every one with an
    # event pair around the call). Event records cost ~10 us of stream time each, so inside the
    # timed region only every 8th step carries one pair (main stream only; <1 % of the region,
    # whatever --steps is) — reported as kernel_ms_in_timed_region, a cross-check.
    k_ev = {k: (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
            for k in range(0, args.steps, 8)}
    s_ev = {}

    # The two halves of a step are independent (the neighbourhood pass works on the trajectory
    # plan, not on the evaluated candidates), so with --overlap 1 they run on two streams, each
    # with its own context ("one context per stream", include/whp.h): the small kernels of
    # whp_eval_swaps fill the SMs that K1 (one warp per scheduler) leaves idle.
    overlap = bool(args.overlap)
    ctx_nb = whp.Context.from_problem(pb, device=local_rank) if overlap else ctx
    main = torch.cuda.current_stream()
    side = torch.cuda.Stream(device=dev, priority=-1) if overlap else main
    fork_ev, join_ev = torch.cuda.Event(), torch.cuda.Event()

    def neighbourhood_half(timed_index):
        s = (it_counter[0] * stride) % (n - Wn + 1)
        if timed_index in s_ev:
            s_ev[timed_index][0].record()
        ctx_nb.eval_swaps(base, s, Wn, dist=sdist, obj=sobj)
        if timed_index in s_ev:
            s_ev[timed_index][1].record()
        ctx_nb.argmin(sobj, sidx)
        ctx_nb.apply_swap(base, s, Wn, sidx)
        it_counter[0] += 1

    def step(timed_index=None):
        if timed_index not in k_ev:
            timed_index = None
        if overlap:
            fork_ev.record(main)
            side.wait_event(fork_ev)
            with torch.cuda.stream(side):
                neighbourhood_half(timed_index)
                join_ev.record(side)
        if timed_index is not None:
            k_ev[timed_index][0].record()
        ctx.eval_candidates(perms, dist=dist, penalty=pen, obj=obj, n_batches=nbat,
                            batch_hash=bhash)
        if timed_index is not None:
            k_ev[timed_index][1].record()
        ctx.argmin(obj, idx, val)
        if overlap:
            main.wait_event(join_ev)
        else:
            neighbourhood_half(timed_index)

    def timed_run():
        sampler = harness.ClockSampler(local_rank, args.clock_period_ms).start().wait_first() if rank == 0 else None
        if sampler:
            sampler.mark()  # warm-up and timed steps are both "under load"
        for _ in range(args.warmup):
            step()
        torch.cuda.synchronize()
        harness.barrier(world)
        launches0 = ctx.launch_count() + (ctx_nb.launch_count() if overlap else 0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for k in range(args.steps):
            step(k)
        e1.record()
        torch.cuda.synchronize()
        harness.barrier(world)
        ms = e0.elapsed_time(e1)
        clocks = sampler.stop() if sampler else None
        return ms, clocks, ctx.launch_count() + (ctx_nb.launch_count() if overlap else 0) - launches0

    ms, clocks, launches = timed_run()
    redo = harness.max_over_ranks(1.0 if (rank == 0 and harness.clocks_rejected(clocks)) else 0.0,
                                  world, dev)
    remeasured = False
    if redo > 0:
        ms, clocks, launches = timed_run()
        remeasured = True
    ms = harness.max_over_ranks(ms, world, dev)
    k_ms_in_region = float(np.mean([a.elapsed_time(b) for a, b in k_ev.values()]))
    k_in_region_samples = len(k_ev)
    k_ev.clear()
    # ---- separate pass: the same step, with an event pair around the evaluation of every step
    for k in range(KERNEL_PASS):
        k_ev[k] = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
        s_ev[k] = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
    torch.cuda.synchronize()
    for k in range(KERNEL_PASS):
        step(k)
    torch.cuda.synchronize()
    k_ms_in_step = float(np.mean([a.elapsed_time(b) for a, b in k_ev.values()]))
    s_ms = float(np.mean([a.elapsed_time(b) for a, b in s_ev.values()]))
    k_ev.clear(), s_ev.clear()
    s_span_ms = s_ms
    # ---- and the evaluation alone on the GPU (nothing on the side stream): under overlap the span
    # above also contains the time K2's blocks wait for SMs the neighbour kernel still holds
    alone_k = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
               for _ in range(KERNEL_PASS)]
    torch.cuda.synchronize()
    for a, b in alone_k:
        a.record()
        ctx.eval_candidates(perms, dist=dist, penalty=pen, obj=obj, n_batches=nbat, batch_hash=bhash)
        b.record()
        ctx.argmin(obj, idx, val)
    torch.cuda.synchronize()
    k_ms = float(np.mean([a.elapsed_time(b) for a, b in alone_k]))
    k_ms_max = harness.max_over_ranks(k_ms, world, dev)
    if overlap:
        # under overlap the events on the side stream span the wait behind K2 as well: the
        # neighbourhood figures come from 50 further iterations of the trajectory run alone
        torch.cuda.synchronize()
        alone = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                 for _ in range(50)]
        for a, b in alone:
            s = (it_counter[0] * stride) % (n - Wn + 1)
            a.record()
            ctx_nb.eval_swaps(base, s, Wn, dist=sdist, obj=sobj)
            b.record()
            ctx_nb.argmin(sobj, sidx)
            ctx_nb.apply_swap(base, s, Wn, sidx)
            it_counter[0] += 1
        torch.cuda.synchronize()
        s_ms = float(np.mean([a.elapsed_time(b) for a, b in alone]))
    ms_per_step = ms / args.steps
    value = n_cand * world / (ms_per_step * 1e-3)

    # ---- sustained: the same step repeated for >= SUSTAIN_S seconds, clocks sampled throughout --
    sustained = None
    if world == 1 and "sustained" in legs:
        n_sus = max(args.steps, int(SUSTAIN_S / (ms_per_step * 1e-3)) + 1)
        sampler = harness.ClockSampler(local_rank, args.clock_period_ms).start().wait_first()
        for _ in range(3):
            step()
        torch.cuda.synchronize()
        sampler.mark()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        for _ in range(n_sus):
            step()
        e1.record()
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        sus_clocks = sampler.stop()
        sus_ms = e0.elapsed_time(e1) / n_sus
        sustained = {"steps": n_sus, "seconds": wall, "ms_per_step": sus_ms,
                     "value": n_cand / (sus_ms * 1e-3), "unit": "candidate plans/s",
                     "vs_timed_region": ms_per_step / sus_ms, "clocks": sus_clocks}

    # ---- end to end through the host-buffer entry point (pinned host memory) ---------------
    e2e = None
    if "e2e" in legs:
        h_dist = torch.zeros(n_cand, dtype=torch.int64).pin_memory()
        h_obj = torch.zeros(n_cand, dtype=torch.float64).pin_memory()
        for _ in range(max(1, min(args.warmup, 2))):
            ctx.eval_candidates_host(h_perms, h_dist, h_obj)
        torch.cuda.synchronize()
        harness.barrier(world)
        e2e_steps = max(1, min(args.steps, 10))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e_idx, e_val = ctx.eval_candidates_host(h_perms, h_dist, h_obj)
        torch.cuda.synchronize()
        e2e_s = harness.max_over_ranks(time.perf_counter() - t0, world, dev)
        harness.barrier(world)
        torch.cuda.synchronize()
        e2e = {"value": n_cand * world * e2e_steps / e2e_s, "unit": "candidate plans/s",
               "h2d_bytes_per_step": int(h_perms.numel() * 4),
               "d2h_bytes_per_step": int(n_cand * 16 + 16),
               "api": "whp_eval_candidates_host (pinned host buffers, chunked copy/compute overlap)",
               "matches_device_path": bool(np.array_equal(h_obj.numpy(), obj.cpu().numpy())
                                           and e_idx == int(idx.item()))}
        # the same through whp_eval_candidates_host16: 16-bit order ids, half the bytes over PCIe
        for _ in range(2):
            ctx.eval_candidates_host(h16, h_dist, h_obj)
        torch.cuda.synchronize()
        harness.barrier(world)
        t0 = time.perf_counter()
        each16 = []
        for _ in range(e2e_steps):
            t1 = time.perf_counter()
            e_idx16, _ = ctx.eval_candidates_host(h16, h_dist, h_obj)  # returns when complete
            each16.append(round((time.perf_counter() - t1) * 1e3, 3))
        torch.cuda.synchronize()
        e16_s = harness.max_over_ranks(time.perf_counter() - t0, world, dev)
        harness.barrier(world)
        e2e["uint16_ids"] = {"value": n_cand * world * e2e_steps / e16_s, "unit": "candidate plans/s",
                             "ms_per_call": each16,
                             "h2d_bytes_per_step": int(h16.numel() * 2),
                             "api": "whp_eval_candidates_host16",
                             "matches_device_path": bool(np.array_equal(h_obj.numpy(), obj.cpu().numpy())
                                                         and e_idx16 == int(idx.item()))}
        del h16, h_perms

    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    nexts, l2_gbs = {}, None
    if "next" in legs:
        # ---- NEXT-1: the NHATC outer loop around the solve, on the device (not part of the step)
        n_outer = 5
        idx_h = torch.zeros(n_outer, dtype=torch.int64, device=dev)
        ctx.nhatc_solve(perms, 1, 1.25, idx_h)  # warm-up (allocates the response scratch)
        torch.cuda.synchronize()
        ev0.record()
        ctx.nhatc_solve(perms, n_outer, 1.25, idx_h)
        ev1.record()
        torch.cuda.synchronize()
        nhatc_ms = ev0.elapsed_time(ev1) / n_outer
        ctx.set_penalty(pb.t, pb.v, pb.w)  # restore the multipliers
        nexts["nhatc_outer_loop"] = {
            "ms_per_outer_iteration": nhatc_ms, "n_outer": n_outer,
            "what": "whp_nhatc_solve: 16,384 plans walked once (D, r), then per outer iteration "
                    "penalty -> argmin -> multiplier update, device only; mean over the call"}

        # ---- NEXT-2: leg sums of the same plans (not part of the step) -------------------------
        leg = torch.zeros(n_cand, dtype=torch.int64, device=dev)
        ctx.eval_legsum(perms, leg)
        torch.cuda.synchronize()
        ev0.record()
        ctx.eval_legsum(perms, leg)
        ev1.record()
        torch.cuda.synchronize()
        legsum_ms = ev0.elapsed_time(ev1)
        nexts["legsum"] = {"ms": legsum_ms, "plans_per_s": n_cand / (legsum_ms * 1e-3),
                           "what": "whp_eval_legsum on the same 16,384 plans (paper-literal Eq. 2)"}

        # ---- NEXT-2, second half: return / largest-gap routing of the same plans ---------------
        nexts["routing"] = {"what": "whp_eval_routing on the same 16,384 plans (readings N5, N6): "
                                    "D and J with the carts routed by the policy"}
        r_obj = torch.zeros(n_cand, dtype=torch.float64, device=dev)
        for pol, pname in ((whp.ROUTE_RETURN, "return"), (whp.ROUTE_LARGEST_GAP, "largest_gap")):
            ctx.eval_routing(perms, pol, leg, r_obj)
            torch.cuda.synchronize()
            ev0.record()
            ctx.eval_routing(perms, pol, leg, r_obj)
            ev1.record()
            torch.cuda.synchronize()
            r_ms = ev0.elapsed_time(ev1)
            nexts["routing"][pname] = {"ms": r_ms, "plans_per_s": n_cand / (r_ms * 1e-3)}

        # ---- NEXT-4: insertion-move neighbourhood of the trajectory plan (not part of the step)
        mW = 128
        mobj = torch.zeros(mW * (mW - 1), dtype=torch.float64, device=dev)
        ctx.eval_moves(base, 0, mW, None, mobj)
        torch.cuda.synchronize()
        ev0.record()
        ctx.eval_moves(base, 0, mW, None, mobj)
        ev1.record()
        torch.cuda.synchronize()
        moves_ms = ev0.elapsed_time(ev1)
        nexts["moves"] = {"ms": moves_ms, "neighbours": mW * (mW - 1),
                          "neighbours_per_s": mW * (mW - 1) / (moves_ms * 1e-3),
                          "what": "whp_eval_moves, all insertion moves of a 128-wide window"}

        # ---- picks actually rescored by one neighbourhood pass (untimed, counted)
        ctx.set_swap_stats(True)
        ctx.eval_swaps(base, 0, Wn, dist=sdist, obj=sobj)
        sw_batches, sw_picks = ctx.get_swap_stats()
        ctx.set_swap_stats(False)
        nexts["rescored"] = {"rescored_batches_per_neighbour": sw_batches / nn,
                             "rescored_picks_per_neighbour": sw_picks / nn,
                             "rescored_picks_per_s": sw_picks / (s_ms * 1e-3)}

        # ---- measured L2 read bandwidth (not in MEASURED_PEAKS.json): 200
        # read-only sweeps of a 32 MB buffer that stays resident in the 126 MB L2, one launch
        l2_gbs = ctx.probe_l2_read(32 << 20, 200)

    peaks = harness.measured_peaks(ROOT)
    counters = harness.ncu_counters(ROOT)

    stress = stress_leg(torch, whp, dev, local_rank, peaks, counters) if (world == 1 and "stress" in legs) else None

    # ---- roofline of the dominant kernel (candidate evaluation) -----------------------------
    bytes_pc = harness.algorithmic_bytes_per_candidate(n, pb.n_items)
    achieved = bytes_pc["survey"] * n_cand / (k_ms_max * 1e-3) / 1e9
    cp = counters.get("paper", {})
    sm_clock_hz = 1e6 * float((clocks or {}).get("sm_mhz") or 1965.0)
    # the units that actually bind the path: warp-instruction issue slots and the
    # shared-memory pipe. Counts per launch come from the ncu capture recorded for these sources
    # (profiles/ncu_counters.csv); the time is this run's; peak = 148 SMs x 4 issue slots (x 1
    # shared-memory wavefront) per clock at the SM clock sampled during the timed region.
    n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    binding = None
    if "warp_inst" in cp and "smem_wavefronts" in cp:
        issue_peak = n_sms * 4 * sm_clock_hz
        smem_peak = n_sms * 1 * sm_clock_hz
        binding = {"issue_slots": {"achieved": cp["warp_inst"] / (k_ms_max * 1e-3), "peak": issue_peak,
                                   "frac": cp["warp_inst"] / (k_ms_max * 1e-3) / issue_peak,
                                   "unit": "warp instructions/s"},
                   "smem_pipe": {"achieved": cp["smem_wavefronts"] / (k_ms_max * 1e-3), "peak": smem_peak,
                                 "frac": cp["smem_wavefronts"] / (k_ms_max * 1e-3) / smem_peak,
                                 "unit": "shared-memory wavefronts/s"},
                   "dram": {"achieved": cp.get("dram_bytes", 0.0) / (k_ms_max * 1e-3) / 1e9,
                            "peak": peaks["hbm_gbs"], "unit": "GB/s",
                            "frac": cp.get("dram_bytes", 0.0) / (k_ms_max * 1e-3) / 1e9 / peaks["hbm_gbs"]},
                   "sm_clock_mhz": sm_clock_hz / 1e6, "counts_from": cp.get("source"),
                   "note": "whole evaluation (K1 + segments + K2), so the fractions average a "
                           "DRAM-streaming kernel and an issue/shared-memory bound one"}
    roofline = {
        "bound": "hbm", "kernel": "whp_eval_candidates (bounds + segments + sets kernels)", "achieved": achieved,
        "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": achieved / peaks["hbm_gbs"],
        "traffic": cp.get("dram_bytes"),
        "traffic_note": (f"ncu dram bytes of one evaluation, captured on these kernel sources "
                         f"({counters['csrc_sha16']}): {cp.get('source')}") if "dram_bytes" in cp else
                        ("no ncu capture recorded for these kernel sources "
                         f"({counters['csrc_sha16']}); see profiles/ for earlier versions"),
        "binding_resource": binding,
        "peak_source": peaks["source"] + ", burst copy figure",
        "bytes_per_candidate": bytes_pc["survey"], "kernel_ms": k_ms_max,
        "kernel_ms_samples": KERNEL_PASS,
        "kernel_ms_how": "mean launch-to-finish time of whp_eval_candidates over a separate pass "
                         "after the timed region, the call alone on the GPU (the timed step runs it "
                         "beside the neighbourhood pass of the other stream)",
        "kernel_ms_span_in_overlapped_step": k_ms_in_step,
        "frac_in_overlapped_step": bytes_pc["survey"] * n_cand / (k_ms_in_step * 1e-3) / 1e9 / peaks["hbm_gbs"],
        "kernel_ms_in_timed_region": k_ms_in_region,
        "kernel_ms_in_timed_region_samples": k_in_region_samples,
        "kernel_share_of_step": k_ms_max / ms_per_step,
        "frac_packed_bytes": bytes_pc["packed"] * n_cand / (k_ms_max * 1e-3) / 1e9 / peaks["hbm_gbs"],
        "frac_hbm_compulsory": bytes_pc["hbm_compulsory"] * n_cand / (k_ms_max * 1e-3) / 1e9 / peaks["hbm_gbs"],
        "l2_read_gbs_measured": l2_gbs,
        "frac_of_l2_read_peak": achieved / l2_gbs if l2_gbs else None,
    }

    if rank != 0:
        return 0
    # ---- CPU baseline: the oracle on a bounded sample, rank 0 at N=1 only -------------------
    cpu = None
    if world == 1 and "cpu" in legs:
        import oracle
        sample = W.perm_rows(wl.seed, n, np.arange(CPU_SAMPLE))
        t0 = time.perf_counter()
        ref = oracle.eval_candidates(pb, sample)
        oracle.argmin(ref["obj"])
        dt = time.perf_counter() - t0
        agree = bool(np.array_equal(ref["obj"], obj[:CPU_SAMPLE].cpu().numpy())
                     and np.array_equal(ref["dist"], dist[:CPU_SAMPLE].cpu().numpy()))
        # the same routine over candidate slices on all host cores (wrapper
        # only: threads around the single-threaded C routine, which runs without the GIL)
        import os
        from concurrent.futures import ThreadPoolExecutor
        ncores = os.cpu_count() or 1
        allrows = W.perm_rows(wl.seed, n, np.arange(n_cand))
        cuts = np.linspace(0, n_cand, 4 * ncores + 1).astype(int)
        t0 = time.perf_counter()
        with ThreadPoolExecutor(ncores) as ex:
            parts = list(ex.map(lambda k: oracle.eval_candidates(pb, allrows[cuts[k]:cuts[k + 1]]),
                                range(4 * ncores)))
        par_obj = np.concatenate([q["obj"] for q in parts])
        oracle.argmin(par_obj)
        dt_par = time.perf_counter() - t0
        agree_all = bool(np.array_equal(par_obj, obj.cpu().numpy()))
        cpu = {"value": CPU_SAMPLE / dt, "unit": "candidate plans/s", "cores": 1,
               "all_cores": {"value": n_cand / dt_par, "cores": ncores, "seconds": dt_par,
                             "sample": "all 16,384 candidates, one thread per core around the "
                                       "same routine",
                             "gpu_results_equal_oracle": agree_all},
               "kind": "oracle", "seconds": dt,
               "sample": f"first {CPU_SAMPLE} of the 16,384 candidates (a1-a5 + argmin), single "
                         "thread, gcc -O2",
               "gpu_results_equal_oracle_on_sample": agree}
    line = {
        "metric": "candidate_plans_per_s", "value": value, "unit": "candidate plans/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64+f64", "data": "synthetic",
        "picks_per_s": value * pb.n_items,
        "config": dict(config_dict(pb, n_cand, world, wl_nb),
                       streams=("candidate evaluation + argmin and neighbourhood pass + argmin + "
                                "apply on two streams, one context each, joined every step")
                       if overlap else "one stream, the calls of a step back to back",
                       k1_warps=args.k1_warps or "library default"),
        "neighbourhood": dict({"ms_per_iteration_eval_swaps": s_ms,
                               "ms_span_on_side_stream_in_step": s_span_ms,
                               "neighbours_per_s": nn / (s_ms * 1e-3),
                               "iterations_per_s": 1.0 / (s_ms * 1e-3)}, **nexts.pop("rescored", {})),
        **nexts,
        "roofline": roofline,
        "sustained": sustained,
        "stress": stress,
        "cpu_baseline": cpu,
        "e2e": e2e,
        "legs": sorted(legs),
        "notes": ["the --impl reference arm (the oracle) re-evaluates every swap neighbour from "
                  "scratch while this arm rescans only the affected batches: the driver's "
                  "ours/reference ratio mixes that algorithmic gain with the hardware's",
                  "roofline.frac is SURVEY.md 8(d)'s nominal gathered bytes against the HBM copy "
                  "peak; roofline.binding_resource gives the units that really bind the path"],
        "gpu_launches": int(launches),
        "clocks": clocks, "remeasured_for_clocks": remeasured,
    }
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--overlap", type=int, default=1, choices=[0, 1],
                    help="1: candidate evaluation and neighbourhood pass of a step on two streams")
    ap.add_argument("--legs", default="all",
                    help="comma list of step,sustained,e2e,next,stress,cpu (default all; profiling "
                         "runs use --legs step or --legs stress)")
    ap.add_argument("--sustain", type=int, default=1, choices=[0, 1],
                    help="1: also repeat the step for >= 2.5 s with the clocks sampled (N=1 only)")
    ap.add_argument("--stress", type=int, default=1, choices=[0, 1],
                    help="1: also time BASELINE.json's stress config at its full 65,536 plans (N=1 only)")
    ap.add_argument("--k1-warps", type=int, default=0, choices=[0, 1, 2, 4, 5],
                    help="warps per block of the boundary kernel (whp_debug_set WHP_DEBUG_K1_WARPS; "
                         "0 = the library's choice): the block-shape table of profiles/r2_head.md")
    ap.add_argument("--clock-period-ms", type=int, default=50,
                    help="nvidia-smi sampling period during the timed region")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)  # timing rule: at least 3 warm-up steps
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
