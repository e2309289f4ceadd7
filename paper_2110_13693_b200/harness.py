"""Host-side measurement helpers used by bench.py (no arithmetic of the method):
candidate sharding across ranks (candidates are independent units, tables
replicated, no data-path collective), max-over-ranks timing, the nvidia-smi clock sampler and
the roofline arithmetic of DESIGN.md §7."""
import json
import os
import subprocess
import threading
import time

THROTTLE_REJECT = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown")


def shard_range(n_total: int, rank: int, world: int):
    """Contiguous candidate range [lo, hi) owned by `rank` (strong scaling of a fixed set)."""
    base, rem = divmod(n_total, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def weak_rows(n_per_rank: int, rank: int):
    """Weak scaling: rank r evaluates candidate ids [r*n, (r+1)*n) of the same seeded stream —
    disjoint across ranks, so the job evaluates world*n distinct plans."""
    return rank * n_per_rank, (rank + 1) * n_per_rank


def dist_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init_dist(backend: str):
    """torch.distributed only for the barrier and the max-over-ranks of the step time."""
    import torch.distributed as dist
    rank, local_rank, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value: float, world: int, device="cpu") -> float:
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, world: int, device="cpu") -> float:
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ---- clocks -----------------------------------------------------------------------------------
_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
          "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
          "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")


class ClockSampler:
    """Samples nvidia-smi every 100 ms on one GPU while the timed region runs."""

    def __init__(self, gpu_index: int = 0, period_ms: int = 100):
        self.gpu_index, self.period_ms = gpu_index, period_ms
        self.proc, self.lines, self.thread = None, [], None
        self.stamps, self.t_mark = [], 0.0

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.gpu_index}", f"--query-gpu={_QUERY}",
                 "--format=csv,noheader,nounits", "-lms", str(self.period_ms)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return self
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())
            self.stamps.append(time.time())

    def wait_first(self, timeout_s: float = 3.0):
        """nvidia-smi takes a few hundred ms to start; wait so short regions get samples."""
        t0 = time.time()
        while self.proc is not None and not self.lines and time.time() - t0 < timeout_s:
            time.sleep(0.02)
        return self

    def mark(self):
        """Samples received from now on count (call when the GPU work starts)."""
        self.t_mark = time.time()

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()  # the exact process we started
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        under_load = [l for l, t in zip(self.lines, self.stamps) if t >= self.t_mark]
        return parse_clock_lines(under_load or self.lines)


def parse_clock_lines(lines) -> dict:
    sm, sm_max, power, reasons = [], [], [], set()
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    for line in lines:
        f = [x.strip() for x in line.split(",")]
        if len(f) < 9:
            continue
        try:
            sm.append(float(f[1]))
            sm_max.append(float(f[2]))
            power.append(float(f[3]))
        except ValueError:
            continue
        for name, val in zip(names, f[5:9]):
            if val.lower() == "active":
                reasons.add(name)
    if not sm:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"], "samples": 0}
    sm_sorted = sorted(sm)
    return {"sm_mhz": sm_sorted[len(sm_sorted) // 2], "sm_max_mhz": max(sm_max),
            "power_w_max": max(power), "reasons": sorted(reasons), "samples": len(sm)}


def clocks_rejected(clocks: dict) -> bool:
    """hw/thermal slowdown, or clocks stuck far below max with no reason (a leftover lock)."""
    if any(r in THROTTLE_REJECT for r in clocks.get("reasons", [])):
        return True
    sm, mx = clocks.get("sm_mhz"), clocks.get("sm_max_mhz")
    if sm and mx and sm < 0.5 * mx and not clocks.get("reasons"):
        return True
    return False


# ---- roofline ----------------------------------------------------------------------------------
def measured_peaks(repo_root: str) -> dict:
    """MEASURED_PEAKS.json (driver-written) or the profiling guide's fallback (6.65 TB/s)."""
    path = os.path.join(repo_root, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": float(p["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json)"}
    except (OSError, KeyError, ValueError):
        return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)"}


def algorithmic_bytes_per_candidate(n_orders: int, n_items: int) -> dict:
    """B = 4 n_orders (perm) + 8 n_orders (order records) + 4 n_items (pick
    records) + 36 (outputs). `packed` counts the 4-byte order records this build really reads;
    `hbm_compulsory` is the part that must come from HBM (the permutation and the outputs)."""
    return {"survey": 4 * n_orders + 8 * n_orders + 4 * n_items + 36,
            "packed": 4 * n_orders + 4 * n_orders + 4 * n_items + 36,
            "hbm_compulsory": 4 * n_orders + 36}


# ---- ncu counters recorded for a given state of the kernels --------------------------------------
EVAL_PATH_SOURCES = ("whp_fast.cu", "whp_eval.cu", "whp_walk.cuh", "whp_internal.cuh")


def csrc_sha16(repo_root: str) -> str:
    """Fingerprint of the sources of the candidate-evaluation kernels (K1, segments, K2, K3 and
    their launcher): counters captured under ncu are only quoted next to a live timing when they
    were captured on these sources."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(repo_root, "paper_2110_13693_b200", "csrc")
    for name in EVAL_PATH_SOURCES:
        with open(os.path.join(csrc, name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def ncu_counters(repo_root: str) -> dict:
    """profiles/ncu_counters.csv: rows `csrc_sha16,workload,counter,value,source` written by hand
    from an `ncu --set full` capture (the .md named in `source` gives the command). Returns
    {workload: {counter: value}} for the rows whose fingerprint matches the sources in the tree,
    plus "stale": True when rows exist but none match."""
    path = os.path.join(repo_root, "profiles", "ncu_counters.csv")
    out, seen = {}, False
    try:
        sha = csrc_sha16(repo_root)
        with open(path) as f:
            for line in f:
                parts = [x.strip() for x in line.split(",")]
                if len(parts) < 5 or parts[0] in ("", "csrc_sha16") or parts[0].startswith("#"):
                    continue
                seen = True
                if parts[0] != sha:
                    continue
                out.setdefault(parts[1], {})[parts[2]] = float(parts[3])
                out[parts[1]]["source"] = parts[4]
    except OSError:
        pass
    out["stale"] = bool(seen and len(out) == 0)
    out["csrc_sha16"] = csrc_sha16(repo_root)
    return out
