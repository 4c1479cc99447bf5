#!/usr/bin/env python
"""bench.py -- one JSON line for the block-matching hot path on B200.

A "step" is one pass of the whole hot path over one synthetic volume pair: variance-based block selection
(S1-S3) followed by exhaustive NCC matching (M1-M5), through the C ABI of libnrr_bm.so (nrr_bm_register: the
selection, the moving-volume statistics and the matching kernels enqueued back to back, no host synchronisation).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                  [--workload tiny|intraop|fullres|highres|batch] [--shard pairs|blocks]

--workload batch: BASELINE.json configs[4], the fullres pair under 32 settings in ONE launch sequence
(nrr_bm_register_batch); value = aggregate blocks/s over the 32 settings.
N > 1 is launched by torch.distributed.run, one rank per GPU.  --shard pairs (default): blocks are independent
(PAPER.md:647-648), every rank matches its own seeded pair, no data-path collective, weak scaling.  --shard blocks:
the paper's own distribution (both images on every processor, the block list distributed): every
rank holds a plan of the same pair, matches a contiguous slice of the canonical block list and the ranks all-gather
16 bytes per block; strong scaling.  Rank 0 prints the line.
--impl reference times the CPU oracle (oracle/) as it stands on the host cores (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from nrr_inputs import CONFIGS, batch_settings, make_pair  # noqa: E402

METRIC = "blocks_per_sec"
UNIT = "blocks/s"
WORKLOADS = sorted(CONFIGS) + ["batch"]
# B200 FP32 (non-tensor) peak derived from the guide's unit counts and clocks:
# 148 SMs x 128 FP32 lanes x 2 flop/FMA x 1.965 GHz
SM_COUNT, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965
FP32_PEAK_TFLOPS = SM_COUNT * FP32_LANES * 2 * SM_MAX_GHZ / 1e3
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "traffic.json")      # DRAM bytes per launch read off kept ncu captures


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="fullres", choices=WORKLOADS)
    ap.add_argument("--shard", default="pairs", choices=["pairs", "blocks"])
    ap.add_argument("--e2e-steps", type=int, default=None, help="steps of the host-buffer (end-to-end) legs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-parity", action="store_true", help="skip the oracle comparison reported under 'parity'")
    ap.add_argument("--option", action="append", default=[], metavar="NAME=VALUE",
                    help="library option for this run (nrr_bm_set_option), e.g. pair_blocks_per_cta=2, force_rows=1, "
                         "disable_tma=1: the A/B runs and sweeps behind DESIGN.md 6.3; recorded under config.options")
    return ap.parse_args(argv)


def parse_options(pairs):
    out = {}
    for item in pairs:
        name, sep, value = item.partition("=")
        if not sep or not name:
            raise SystemExit("--option wants NAME=VALUE, got %r" % item)
        out[name] = float(value)
    return out


def valid_candidates(blocks: np.ndarray, dims, block, window) -> np.ndarray:
    """Candidates per block that survive the skip rule (pure geometry; used only to count useful FMAs)."""
    out = np.ones(len(blocks), dtype=np.int64)
    for a in range(3):
        o = blocks[:, a].astype(np.int64) - (block[a] - 1) // 2
        lo = np.maximum(-window[a], -o)
        hi = np.minimum(window[a], dims[a] - block[a] - o)
        out *= (hi - lo + 1)
    return out


def rank_config(cfg, rank: int):
    """--shard pairs: every rank matches its OWN seeded pair (independent units)."""
    import dataclasses
    return dataclasses.replace(cfg, seed=cfg.seed + 17 * rank)


def shard_range(n: int, rank: int, world: int):
    """--shard blocks: rank r's contiguous slice [first, first + count) of the canonical (z-major) block list."""
    first = (n * rank) // world
    return first, (n * (rank + 1)) // world - first


def exchange_block_results(dist, o_disp, o_ncc, n_all: int, rank: int, world: int, send, recv):
    """--shard blocks: the one data-path collective, an all-gather of 16 bytes per block (dx, dy, dz, NCC bits).
    o_disp [n_all][3] int32 / o_ncc [n_all] fp32 hold this rank's slice on entry and every rank's on return;
    send [cmax][4] / recv [world][cmax][4] int32 are scratch (cmax = the largest slice)."""
    import torch
    first, count = shard_range(n_all, rank, world)
    send[:count, :3] = o_disp[first:first + count]
    send[:count, 3] = o_ncc[first:first + count].view(torch.int32)
    dist.all_gather_into_tensor(recv.view(-1, 4), send)
    for r in range(world):
        f_r, c_r = shard_range(n_all, r, world)
        o_disp[f_r:f_r + c_r] = recv[r, :c_r, :3]
        o_ncc[f_r:f_r + c_r] = recv[r, :c_r, 3].view(torch.float32)


def reduce_over_ranks(total_ms: float, units: float, world: int, device=None, dist=None):
    """Whole-job figures: time = MAX over ranks, units = SUM over ranks (the only collectives of --shard pairs)."""
    import torch
    t = torch.tensor([float(total_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, device_index: int, period_s: float = 0.01):
        super().__init__(daemon=True)
        self.period = period_s
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                uuid = "GPU-" + str(torch.cuda.get_device_properties(device_index).uuid)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    _NAMES = {
        0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
        0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost",
    }

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                mhz = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.samples.append(mhz)
                for bit, name in self._NAMES.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        med = statistics.median(self.samples) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------ the oracle legs
def workload_settings(name):
    """[(block, stride, window, frac)] of a workload, and the Config that generates its volume pair."""
    if name == "batch":
        return [(s.block, s.stride, s.window, s.frac) for s in batch_settings()], CONFIGS["fullres"]
    c = CONFIGS[name]
    return [(c.block, c.stride, c.window, c.frac)], c


def oracle_step(oracle, settings, fixed, moving, mask, budget_blocks, nthreads=0):
    """One oracle step over `settings`: the full selection of each, and the matching of at most `budget_blocks` evenly
    spaced selected blocks per setting (None: every block).  Selection and matching are timed separately so that a
    sampled step can be scaled to the whole one: est = t_select + sum_s t_match_s * n_s / n_sample_s."""
    t_select = 0.0
    per = []
    for block, stride, window, frac in settings:
        t0 = time.perf_counter()
        sel = oracle.select(fixed, block, stride, frac, mask)
        t1 = time.perf_counter()
        n = len(sel["centres"])
        k = n if budget_blocks is None else min(n, max(1, int(budget_blocks)))
        idx = np.arange(n) if k == n else np.unique(np.linspace(0, n - 1, k).astype(np.int64))
        res = oracle.match(fixed, moving, sel["centres"][idx], block, window, nthreads=nthreads)
        t2 = time.perf_counter()
        t_select += t1 - t0
        per.append({"n": n, "n_sample": len(idx), "t_match": t2 - t1, "evals": int(res["nvalid"].sum())})
    n_all = sum(p["n"] for p in per)
    est_match = sum(p["t_match"] * p["n"] / max(1, p["n_sample"]) for p in per)
    return {"n": n_all, "n_sample": sum(p["n_sample"] for p in per), "t_select": t_select,
            "t_match": sum(p["t_match"] for p in per), "est_step": t_select + est_match,
            "evals": sum(p["evals"] for p in per), "sampled": any(p["n_sample"] < p["n"] for p in per)}


def oracle_budget(oracle, settings, fixed, moving, mask, seconds):
    """Blocks per setting that keep one oracle step near `seconds` of wall time (None: the whole step fits)."""
    r = oracle_step(oracle, settings, fixed, moving, mask, 8)          # also pages in and spins up the threads
    if r["est_step"] <= seconds:
        return None
    per_block = max(1e-9, r["t_match"] / max(1, r["n_sample"]))
    return max(8, int((seconds - min(seconds * 0.5, r["t_select"])) / per_block / len(settings)))


def run_reference(args, rank):
    """The reference arm of this tier is the CPU oracle, as it stands, on the host cores (rank 0 only).  Every step is
    the WHOLE oracle step when it fits a few seconds (tiny, intraop, fullres); otherwise (highres, batch) the full
    selection plus a bounded sample of blocks, scaled to the whole step exactly as `cpu_baseline` does."""
    if rank != 0:
        return
    import oracle
    settings, cfg = workload_settings(args.workload)
    fixed, moving, mask = make_pair(cfg)
    cores = oracle.max_threads()
    warm = max(1, min(args.warmup, 2))
    budget = oracle_budget(oracle, settings, fixed, moving, mask, 6.0)
    for _ in range(warm):
        oracle_step(oracle, settings, fixed, moving, mask, budget)
    steps = max(1, min(args.steps, 10))
    total, blocks, evals, t_sel, t_match, n_sample = 0.0, 0, 0.0, 0.0, 0.0, 0
    for _ in range(steps):
        r = oracle_step(oracle, settings, fixed, moving, mask, budget)
        total += r["est_step"]
        blocks += r["n"]
        evals += r["evals"] * (r["n"] / max(1, r["n_sample"]))
        t_sel, t_match, n_sample, sampled, n_step = r["t_select"], r["t_match"], r["n_sample"], r["sampled"], r["n"]
    value = blocks / total
    sample = ("each step = the whole oracle step (full selection + matching of all %d blocks)" % n_step) if not sampled else (
        "each step = full selection (%.3f s) + matching of %d of %d evenly spaced selected blocks (%.2f s), scaled to the "
        "whole step" % (t_sel, n_sample, n_step, t_match))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0, "steps": steps,
        "warmup": warm, "ms_per_step": 1e3 * total / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_of(args.workload, cfg, settings),
        "cand_evals_per_sec": evals / total,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def config_of(workload, cfg, settings):
    c = {"workload": workload, "dims": list(cfg.dims)}
    if workload == "batch":
        c.update({"settings": len(settings), "block": "{5,7,9,11}^3", "stride": [5, 5, 5], "window": "+-{3,5,7,9}", "frac": "{0.1,0.3}"})
    else:
        c.update({"block": list(cfg.block), "stride": list(cfg.stride), "window": list(cfg.window), "frac": cfg.frac})
    return c


def parity_report(oracle, settings, fixed, moving, mask, results, budget_blocks):
    """GPU results against the oracle, outside every timed region (north_star: 'counted and reported').
    results[s] = (blocks, disp, ncc) numpy arrays trimmed to K."""
    out = {"exempt_ties": 0, "blocks_in_tie_band": 0, "disp_mismatch_outside_band": 0, "max_abs_dncc": 0.0,
           "selection_equal": True, "blocks_checked": 0, "blocks": 0}
    for (block, stride, window, frac), (gb, gd, gs) in zip(settings, results):
        sel = oracle.select(fixed, block, stride, frac, mask)
        same = len(gb) == len(sel["centres"]) and np.array_equal(gb, sel["centres"])
        out["selection_equal"] = bool(out["selection_equal"] and same)
        out["blocks"] += int(len(gb))
        if not same:
            continue
        n = len(gb)
        k = n if budget_blocks is None else min(n, max(1, int(budget_blocks)))
        idx = np.arange(n) if k == n else np.unique(np.linspace(0, n - 1, k).astype(np.int64))
        ora = oracle.match(fixed, moving, sel["centres"][idx], block, window)
        differ = np.any(gd[idx] != ora["disp"], axis=1)
        band = ora["gap"] < 1e-5
        out["exempt_ties"] += int((differ & band).sum())
        out["blocks_in_tie_band"] += int(band.sum())
        out["disp_mismatch_outside_band"] += int((differ & ~band).sum())
        if len(idx):
            out["max_abs_dncc"] = max(out["max_abs_dncc"], float(np.max(np.abs(gs[idx].astype(np.float64) - ora["ncc"]))))
        out["blocks_checked"] += int(len(idx))
    out["tolerances"] = {"disp": "bit-exact outside oracle top-two gap < 1e-5", "ncc_abs": 1e-4}
    out["ok"] = bool(out["selection_equal"] and out["disp_mismatch_outside_band"] == 0 and out["max_abs_dncc"] <= 1e-4)
    return out


def traffic_for(kernel: str, workload: str):
    """DRAM bytes per launch of `kernel` on `workload` from a kept `ncu --set full` capture (profiles/traffic.json:
    {"<kernel>@<workload>": {"bytes": ..., "file": "profiles/..."}}); None when no capture of that kernel exists."""
    try:
        with open(TRAFFIC_FILE) as fh:
            e = json.load(fh).get("%s@%s" % (kernel, workload))
        return (int(e["bytes"]), e.get("file")) if e else (None, None)
    except Exception:
        return None, None


class CudaBackend:
    """The real thing: cuda:<local_rank>, the product library, CUDA events.  (tests/test_bench_dryrun.py passes a
    stand-in with the same five members to run main() end to end on the CPU emulation of the kernels.)"""

    flush_bytes = 256 * 1024 * 1024          # > 126 MB L2
    collective_backend = "nccl"

    def __init__(self, local_rank: int):
        import torch
        import paper_2308_10868_b200 as nrr
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
        nrr.lib()
        torch.cuda.set_device(local_rank)
        self.nrr = nrr
        self.dev = torch.device("cuda", local_rank)

    def sync(self):
        import torch
        torch.cuda.synchronize()

    def event(self):
        import torch
        return torch.cuda.Event(enable_timing=True)

    def stream(self):
        import torch
        return torch.cuda.current_stream()

    def pin(self, t):
        return t.pin_memory()


def main(argv=None, backend_factory=CudaBackend):
    args = parse_args(argv)
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist

    be = backend_factory(local_rank)
    nrr, dev = be.nrr, be.dev
    options = parse_options(args.option)
    for name, value in options.items():
        nrr.nrr_bm_set_option(name, value)
    if world > 1:
        dist.init_process_group(be.collective_backend, device_id=dev if dev.type == "cuda" else None)
    shard_blocks = args.shard == "blocks" and world > 1
    if shard_blocks and args.workload == "batch":
        raise SystemExit("--shard blocks distributes ONE block list; the batch workload has 32")

    settings, base_cfg = workload_settings(args.workload)
    cfg = base_cfg if shard_blocks else rank_config(base_cfg, rank)      # blocks mode: the same pair on every rank
    dims = cfg.dims
    fixed_h, moving_h, mask_h = make_pair(cfg)
    fixed = torch.from_numpy(fixed_h).to(dev)
    moving = torch.from_numpy(moving_h).to(dev)
    mask = torch.from_numpy(mask_h).to(dev) if mask_h is not None else None
    flush = torch.empty(be.flush_bytes // 4, dtype=torch.float32, device=dev)      # 256 MB > 126 MB L2
    stream = be.stream()
    is_batch = args.workload == "batch"
    block, stride, window, frac = settings[0]

    def barrier():
        be.sync()
        if world > 1:
            dist.barrier()
        be.sync()

    # ---- the step
    plan = None
    if is_batch:
        st_objs = list(batch_settings())
        holder = {}

        def step():
            holder["res"], holder["n"] = nrr.nrr_bm_register_batch(fixed, moving, st_objs, mask)

        def results():
            ns = holder["n"].cpu().numpy()
            return [(b[:k].cpu().numpy(), d[:k].cpu().numpy(), s[:k].cpu().numpy()) for (b, d, s), k in zip(holder["res"], ns)]
    elif shard_blocks:
        # both images on every processor, the block list distributed.  Pre-operative: every rank
        # builds the same plan.  A step = this rank's slice of the block list + the exchange of 16 bytes per block.
        plan = nrr.nrr_bm_plan_create(fixed, block, stride, window, frac, mask)
        n_all = plan.n
        first, count = shard_range(n_all, rank, world)
        o_disp = torch.zeros((n_all, 3), dtype=torch.int32, device=dev)
        o_ncc = torch.zeros((n_all,), dtype=torch.float32, device=dev)
        cmax = max(shard_range(n_all, r, world)[1] for r in range(world))
        send = torch.zeros((cmax, 4), dtype=torch.int32, device=dev)            # (dx, dy, dz, ncc bits): 16 B per block
        recv = torch.zeros((world, cmax, 4), dtype=torch.int32, device=dev)

        def step():
            nrr.nrr_bm_plan_match_range(plan, moving, o_disp, o_ncc, first=first, count=count)
            exchange_block_results(dist, o_disp, o_ncc, n_all, rank, world, send, recv)

        def results():
            return [(nrr.nrr_bm_plan_blocks_host(plan), o_disp.cpu().numpy(), o_ncc.cpu().numpy())]
    else:
        cap = max(1, nrr.nrr_bm_capacity_bound(dims, block, stride, frac)[1])      # the library's own count rule
        o_blocks = torch.empty((cap, 3), dtype=torch.int32, device=dev)
        o_disp = torch.empty((cap, 3), dtype=torch.int32, device=dev)
        o_ncc = torch.empty((cap,), dtype=torch.float32, device=dev)
        o_n = torch.zeros((), dtype=torch.int32, device=dev)

        def step():
            nrr.nrr_bm_register(fixed, moving, block, stride, window, frac, mask, capacity=cap,
                                out_blocks=o_blocks, out_n=o_n, out_disp=o_disp, out_ncc=o_ncc)

        def results():
            k = int(o_n.item())
            return [(o_blocks[:k].cpu().numpy(), o_disp[:k].cpu().numpy(), o_ncc[:k].cpu().numpy())]

    def warm_up():
        for _ in range(args.warmup):
            flush.zero_()
            step()
        nrr.nrr_bm_check_async_error()
        return results()

    # ---- warm-up, then parity against the oracle BEFORE anything is timed (north_star: parity is the first gate).
    # If the default kernels' results are wrong on this GPU (they were written while no hardware was reachable,
    # DESIGN.md section 11) the run falls back, loudly, to the kernels measured in round 1 -- never to the CPU.
    parity, kernel_fallback = None, None
    pb = None if args.workload in ("tiny", "intraop", "fullres") else (400 if args.workload == "highres" else 24)
    try:
        res = warm_up()
        if not args.no_parity and rank == 0:
            import oracle
            parity = parity_report(oracle, settings, fixed_h, moving_h, mask_h, res, pb)
        failed = parity is not None and not parity["ok"]
        why = "parity against the oracle failed: %s" % json.dumps(parity) if failed else None
    except nrr.NrrError as e:
        failed, why = True, "the default kernels raised %s" % e
    if world > 1:      # every rank must take the same path
        flag = torch.tensor([1.0 if failed else 0.0], dtype=torch.float64, device=dev)
        dist.all_reduce(flag, op=dist.ReduceOp.MAX)
        failed = bool(flag.item() > 0)
    if failed:
        print("bench.py: falling back to the round-1 kernels: %s" % why, file=sys.stderr)
        for name in ("force_rows", "boxstat_generic", "select_generic"):
            nrr.nrr_bm_set_option(name, 1)
        kernel_fallback = why or "another rank failed"
        res = warm_up()
        if not args.no_parity and rank == 0:
            import oracle
            parity = parity_report(oracle, settings, fixed_h, moving_h, mask_h, res, pb)
    n = sum(len(r[0]) for r in res)                                     # blocks per step on this rank's pair
    valid_per = [valid_candidates(r[0], dims, s[0], s[2]) for r, s in zip(res, settings)]
    useful_fma_per = [int(v.sum()) * s[0][0] * s[0][1] * s[0][2] for v, s in zip(valid_per, settings)]
    useful_fma = sum(useful_fma_per)
    evals = float(sum(int(v.sum()) for v in valid_per))

    # ---- timed region: device-resident inputs, CUDA events on the launching stream, L2 flushed between steps
    sampler = ClockSampler(local_rank)
    sampler.start()
    nrr.nrr_bm_profile_enable(True)
    nrr.nrr_bm_profile_read()
    nrr.nrr_bm_launch_count(reset=True)
    ev = [(be.event(), be.event()) for _ in range(args.steps)]
    barrier()
    for i in range(args.steps):
        flush.zero_()
        ev[i][0].record(stream)
        step()
        ev[i][1].record(stream)
    barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    launches = nrr.nrr_bm_launch_count(reset=True)
    prof = nrr.nrr_bm_profile_read()
    nrr.nrr_bm_profile_enable(False)
    clocks = sampler.stop()
    total_ms = float(sum(step_ms))
    units = float(n) * args.steps / (world if shard_blocks else 1)      # blocks mode: the ranks share ONE block list
    total_ms_max, blocks_all = reduce_over_ranks(total_ms, units, world, dev, dist)
    value = blocks_all / (total_ms_max * 1e-3)

    # ---- end-to-end legs: the same work through the host-buffer C-ABI calls, copies inside the timed region
    e2e_steps = args.e2e_steps if args.e2e_steps is not None else max(3, min(args.steps, 30))
    fixed_p = be.pin(torch.from_numpy(fixed_h))
    moving_p = be.pin(torch.from_numpy(moving_h))
    mask_p = be.pin(torch.from_numpy(mask_h)) if mask_h is not None else None
    e2e = None
    if is_batch:
        # no host form of the sweep: pinned volumes go up with torch copies, every setting's results come back
        def e2e_step():
            f = fixed_p.to(dev, non_blocking=True)
            m = moving_p.to(dev, non_blocking=True)
            k = mask_p.to(dev, non_blocking=True) if mask_p is not None else None
            r, ns = nrr.nrr_bm_register_batch(f, m, st_objs, k)
            ns_h = ns.cpu()
            return sum(int(v) for v in ns_h), [(b.cpu(), d.cpu(), s.cpu()) for (b, d, s) in r]
        h2d = fixed_h.nbytes + moving_h.nbytes + (mask_h.nbytes if mask_h is not None else 0)
        d2h_of = lambda: sum(b.numel() * 4 + d.numel() * 4 + s.numel() * 4 for (b, d, s) in holder["res"]) + 4 * len(settings)
    else:
        cap_h = max(1, nrr.nrr_bm_capacity_bound(dims, block, stride, frac)[1])
        ob = be.pin(torch.empty((cap_h, 3), dtype=torch.int32))
        od = be.pin(torch.empty((cap_h, 3), dtype=torch.int32))
        on = be.pin(torch.empty((cap_h,), dtype=torch.float32))

        def e2e_step():
            rb, rd, rs = nrr.nrr_bm_register_host(fixed_p, moving_p, block, stride, window, frac, mask_p, ob, od, on)
            return len(rb), rd
        h2d = fixed_h.nbytes + moving_h.nbytes + (mask_h.nbytes if mask_h is not None else 0)
        d2h_of = lambda: int(n) * (12 + 12 + 4) + 4
    for _ in range(3):
        e2e_step()
    barrier()
    e2e_t, e2e_n = 0.0, 0
    for _ in range(e2e_steps):
        flush.zero_()
        be.sync()
        t0 = time.perf_counter()
        k, last = e2e_step()
        be.sync()
        e2e_t += time.perf_counter() - t0
        e2e_n += k
    barrier()
    e2e_t_max, e2e_blocks = reduce_over_ranks(e2e_t, float(e2e_n), world, dev, dist)
    if not is_batch:
        assert np.array_equal(np.asarray(last), res[0][1]), "host and device forms disagree"
    e2e = {"value": e2e_blocks / e2e_t_max, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h_of(),
           "steps": e2e_steps, "ms_per_step": 1e3 * e2e_t_max / e2e_steps,
           "call": "torch pinned copies + nrr_bm_register_batch" if is_batch else "nrr_bm_register_host (pre- and intra-operative work, both volumes uploaded)"}
    # plan form: the pre-operative half is done once; a step uploads the intra-operative volume only
    if not is_batch:
        try:      # a secondary leg: on one GPU its failure is reported in the line, it does not cost the line
            hplan = nrr.nrr_bm_plan_create_host(fixed_p, block, stride, window, frac, mask_p)
            pd = be.pin(torch.empty((hplan.n, 3), dtype=torch.int32))
            pn = be.pin(torch.empty((hplan.n,), dtype=torch.float32))
            for _ in range(3):
                nrr.nrr_bm_plan_match_host(hplan, moving_p, pd, pn)
            barrier()
            t_plan = 0.0
            for _ in range(e2e_steps):
                flush.zero_()
                be.sync()
                t0 = time.perf_counter()
                nrr.nrr_bm_plan_match_host(hplan, moving_p, pd, pn)
                t_plan += time.perf_counter() - t0
            barrier()
            assert np.array_equal(np.asarray(pd), res[0][1]), "plan and register forms disagree"
            t_plan_max, plan_blocks = reduce_over_ranks(t_plan, float(hplan.n) * e2e_steps, world, dev, dist)
            e2e["plan"] = {"value": plan_blocks / t_plan_max, "unit": UNIT, "ms_per_step": 1e3 * t_plan_max / e2e_steps,
                           "h2d_bytes_per_step": moving_h.nbytes, "d2h_bytes_per_step": int(hplan.n) * 16,
                           "call": "nrr_bm_plan_match_host (intra-operative work only; selection and fixed-block records "
                                   "were made by nrr_bm_plan_create_host before the timed region)"}
            nrr.nrr_bm_plan_destroy(hplan)
        except Exception as e:
            if world > 1:
                raise
            e2e["plan"] = {"error": repr(e)}
    if plan is not None:
        nrr.nrr_bm_plan_destroy(plan)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (matching): useful FMAs / its own average launch duration
    match_calls = max(1, prof["match_calls"])
    match_ms = prof["match_ms"] / match_calls
    launch_fma = useful_fma / len(settings) / (world if shard_blocks else 1)      # average matching launch
    achieved_tflops = 2.0 * launch_fma / (match_ms * 1e-3) / 1e12
    if is_batch:      # the 32 matching launches overlap on several streams: their spans are not additive -- use the step
        achieved_tflops = 2.0 * useful_fma / (total_ms / args.steps * 1e-3) / 1e12
    peak_measured, micro = None, None
    try:
        peak_measured = nrr.nrr_bm_fp32_peak()
        micro = nrr.nrr_bm_fp32_microbench() if hasattr(nrr, "nrr_bm_fp32_microbench") else None
    except Exception as e:  # pragma: no cover
        print("fp32 microbenchmark failed: %s" % e, file=sys.stderr)
    # the launch shape depends on the number of blocks the launch is SIZED for: this rank's slice (--shard blocks), or
    # the capacity bound of nrr_bm_register (K is known only on the device; CTAs beyond K exit at once)
    launch_n = count if shard_blocks else (int(len(res[0][0])) if is_batch else cap)
    info = nrr.nrr_bm_match_info(dims, block, window, int(launch_n))
    kernel_name = {2: "match_pair_kernel", 1: "match_rows_kernel", 0: "match_generic_kernel"}[info["kernel"]]
    traffic, traffic_file = traffic_for(kernel_name, args.workload)
    roofline = {
        "bound": "alu", "kernel": kernel_name if not is_batch else "match_pair_kernel (32 launches, all shapes)",
        "launch": {"threads": info["threads"], "smem_bytes": info["smem_bytes"],
                   "blocks_per_cta": info["blocks_per_cta"], "tma": info["tma"], "sized_for_blocks": int(launch_n)},
        "achieved": achieved_tflops, "peak": FP32_PEAK_TFLOPS,
        "unit": "TFLOP/s", "frac": achieved_tflops / FP32_PEAK_TFLOPS,
        "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (MEASURED_PEAKS.json has no FP32 figure)",
        "peak_measured_ffma": peak_measured,
        "frac_of_measured_ffma": (achieved_tflops / peak_measured) if peak_measured else None,
        "microbench_tflops": micro,
        "traffic": traffic, "traffic_source": traffic_file or "no ncu --set full capture of this kernel on this workload is kept under profiles/",
        "useful_fma_per_launch": launch_fma, "kernel_ms": match_ms,
    }

    # ---- the oracle, as it stands, on this box's host cores (a reported baseline, not the target)
    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        import oracle
        budget = oracle_budget(oracle, settings, fixed_h, moving_h, mask_h, 15.0)          # ~15 s of CPU work
        r = oracle_step(oracle, settings, fixed_h, moving_h, mask_h, budget)
        rate_all = r["n_sample"] / max(r["t_match"], 1e-9)
        # the same matching on ONE thread, on a sample sized for ~4 s: the measured 1 -> all-thread scaling
        nt = oracle.max_threads()
        b1 = max(4, int(4.0 * rate_all / max(1, nt) / len(settings)))
        r1 = oracle_step(oracle, settings, fixed_h, moving_h, mask_h, b1, nthreads=1)
        rate_1 = r1["n_sample"] / max(r1["t_match"], 1e-9)
        est1 = r1["t_select"] + sum([r1["t_match"] * r1["n"] / max(1, r1["n_sample"])])
        cpu_baseline = {
            "value": r["n"] / r["est_step"], "unit": UNIT, "cores": nt, "kind": "oracle",
            "sample": ("the whole step: full selection (%.3f s) + matching of all %d blocks (%.2f s)" % (r["t_select"], r["n"], r["t_match"]))
            if not r["sampled"] else
            ("full selection (%.3f s) + matching of %d of %d evenly spaced selected blocks (%.2f s), scaled to the whole "
             "step" % (r["t_select"], r["n_sample"], r["n"], r["t_match"])),
            "cand_evals_per_sec": r["evals"] / max(r["t_match"], 1e-9),
            "threads_1_value": r1["n"] / est1,
            "threads_1_sample": "matching of %d blocks on one thread (%.2f s)" % (r1["n_sample"], r1["t_match"]),
            "matching_scaling_1_to_all_threads": rate_all / rate_1,
        }

    ms_per_step = total_ms_max / args.steps

    def per_call(key):
        return prof[key + "_ms"] / max(1, prof[key + "_calls"])
    sel_ms = prof["select_ms"] / args.steps
    stats_ms = prof["moving_stats_ms"] / args.steps
    prep_ms = prof["prep_ms"] / args.steps
    match_total_ms = prof["match_ms"] / args.steps
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if shard_blocks else "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": dict(config_of(args.workload, cfg, settings), blocks_per_pair=int(n),
                       candidates_per_block=cfg.n_candidates if not is_batch else "343..6859",
                       l2="flushed between steps (256 MB write)", options=options,
                       parallelism=("block list sharded over ranks + all-gather of 16 B/block" if shard_blocks else "independent pairs per GPU")),
        "cand_evals_per_sec": evals * args.steps * (1 if shard_blocks else world) / (total_ms_max * 1e-3),
        # only matching is time-critical: the two halves are reported separately and summed
        "ms_per_volume_pair": {"select": sel_ms + prep_ms, "match": stats_ms + match_total_ms, "sum": sel_ms + prep_ms + stats_ms + match_total_ms,
                               "step_wall": ms_per_step,
                               "note": "per step, from CUDA-event spans inside the library; select = S1-S3 + fixed-block records "
                                       "(pre-operative), match = M2 + M1/M3-M5 (intra-operative); moving statistics overlap the "
                                       "selection on a side stream, so the sum can exceed step_wall"},
        "phase_ms": {"select": per_call("select"), "moving_stats": per_call("moving_stats"),
                     "fixed_records": per_call("prep"), "match": match_ms,
                     "calls_per_step": {k: prof[k + "_calls"] / args.steps for k in ("select", "moving_stats", "prep", "match")}},
        "match_only": {"blocks_per_sec": n / (world if shard_blocks else 1) / (match_total_ms * 1e-3),
                       "cand_evals_per_sec": evals / (world if shard_blocks else 1) / (match_total_ms * 1e-3)},
        "fp32_peak_frac": achieved_tflops / FP32_PEAK_TFLOPS,
        "roofline": roofline,
        "parity": parity,
        "kernel_fallback": kernel_fallback,
        "cpu_baseline": cpu_baseline,
        "e2e": e2e,
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
