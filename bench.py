#!/usr/bin/env python
"""bench.py -- one JSON line for the block-matching hot path on B200.

A "step" is one pass of the whole hot path over one synthetic volume pair: variance-based block selection
(S1-S3) followed by exhaustive NCC matching (M1-M5), through the C ABI of libnrr_bm.so (nrr_bm_register: the
selection, the moving-volume statistics and the matching kernels enqueued back to back, no host synchronisation).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload fullres]

N > 1 is launched by torch.distributed.run, one rank per GPU; blocks are independent, so
every rank matches its own seeded pair (weak scaling, no data-path collective) and rank 0 prints the line.
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

from nrr_inputs import CONFIGS, make_pair  # noqa: E402

METRIC = "blocks_per_sec"
UNIT = "blocks/s"
# B200 FP32 (non-tensor) peak derived from the guide's unit counts and clocks:
# 148 SMs x 128 FP32 lanes x 2 flop/FMA x 1.965 GHz
SM_COUNT, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965
FP32_PEAK_TFLOPS = SM_COUNT * FP32_LANES * 2 * SM_MAX_GHZ / 1e3


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="fullres", choices=sorted(CONFIGS))
    ap.add_argument("--e2e-steps", type=int, default=None, help="steps of the host-buffer (end-to-end) leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args(argv)


def valid_candidates(blocks: np.ndarray, cfg) -> np.ndarray:
    """Candidates per block that survive the skip rule (pure geometry; used only to count useful FMAs)."""
    out = np.ones(len(blocks), dtype=np.int64)
    for a in range(3):
        o = blocks[:, a].astype(np.int64) - (cfg.block[a] - 1) // 2
        lo = np.maximum(-cfg.window[a], -o)
        hi = np.minimum(cfg.window[a], cfg.dims[a] - cfg.block[a] - o)
        out *= (hi - lo + 1)
    return out


def rank_config(cfg, rank: int):
    """Every rank matches its OWN seeded pair (independent units): no data-path collective."""
    import dataclasses
    return dataclasses.replace(cfg, seed=cfg.seed + 17 * rank)


def reduce_over_ranks(total_ms: float, units: float, world: int, device=None, dist=None):
    """Whole-job figures: time = MAX over ranks, units = SUM over ranks (the only collectives of the run)."""
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


def oracle_step(oracle, cfg, fixed, moving, mask, sample_blocks):
    """One bounded oracle step: full selection + matching of `sample_blocks` evenly spaced selected blocks."""
    t0 = time.perf_counter()
    sel = oracle.select(fixed, cfg.block, cfg.stride, cfg.frac, mask)
    t1 = time.perf_counter()
    n = len(sel["centres"])
    idx = np.unique(np.linspace(0, n - 1, min(sample_blocks, n)).astype(np.int64))
    res = oracle.match(fixed, moving, sel["centres"][idx], cfg.block, cfg.window)
    t2 = time.perf_counter()
    return {"n": n, "n_sample": len(idx), "t_select": t1 - t0, "t_match": t2 - t1, "evals": int(res["nvalid"].sum())}


def run_reference(args, rank):
    """The reference arm of this tier is the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import oracle
    cfg = CONFIGS[args.workload]
    fixed, moving, mask = make_pair(cfg)
    cores = oracle.max_threads()
    sample = 256
    for _ in range(max(1, min(args.warmup, 2))):
        oracle_step(oracle, cfg, fixed, moving, mask, 32)
    times, blocks, evals = [], 0, 0
    steps = max(1, min(args.steps, 20))
    for _ in range(steps):
        r = oracle_step(oracle, cfg, fixed, moving, mask, sample)
        times.append(r["t_select"] + r["t_match"])
        blocks += r["n_sample"]
        evals += r["evals"]
    total = sum(times)
    value = blocks / total
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0, "steps": steps,
        "warmup": max(1, min(args.warmup, 2)), "ms_per_step": 1e3 * total / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "dims": list(cfg.dims), "block": list(cfg.block),
                   "stride": list(cfg.stride), "window": list(cfg.window), "frac": cfg.frac},
        "cand_evals_per_sec": evals / total,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "each step = full selection + matching of %d evenly spaced selected blocks" % sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


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
    if world > 1:
        dist.init_process_group(be.collective_backend, device_id=dev if dev.type == "cuda" else None)

    cfg = rank_config(CONFIGS[args.workload], rank)
    fixed_h, moving_h, mask_h = make_pair(cfg)
    fixed = torch.from_numpy(fixed_h).to(dev)
    moving = torch.from_numpy(moving_h).to(dev)
    mask = torch.from_numpy(mask_h).to(dev) if mask_h is not None else None
    flush = torch.empty(be.flush_bytes // 4, dtype=torch.float32, device=dev)      # 256 MB > 126 MB L2
    stream = be.stream()

    ngrid = 1
    for a in range(3):
        ngrid *= (cfg.dims[a] - cfg.block[a]) // cfg.stride[a] + 1
    cap = max(1, min(ngrid, int(np.floor(0.5 + ngrid * cfg.frac))))      # host-side upper bound on K
    o_blocks = torch.empty((cap, 3), dtype=torch.int32, device=dev)
    o_disp = torch.empty((cap, 3), dtype=torch.int32, device=dev)
    o_ncc = torch.empty((cap,), dtype=torch.float32, device=dev)
    o_n = torch.zeros((), dtype=torch.int32, device=dev)

    def step():
        nrr.nrr_bm_register(fixed, moving, cfg.block, cfg.stride, cfg.window, cfg.frac, mask, capacity=cap,
                            out_blocks=o_blocks, out_n=o_n, out_disp=o_disp, out_ncc=o_ncc)

    def barrier():
        be.sync()
        if world > 1:
            dist.barrier()
        be.sync()

    for _ in range(args.warmup):
        flush.zero_()
        step()
    nrr.nrr_bm_check_async_error()
    n = int(o_n.item())
    blocks, disp, ncc = o_blocks[:n], o_disp[:n], o_ncc[:n]
    valid = valid_candidates(blocks.cpu().numpy(), cfg)
    nvox_block = cfg.block[0] * cfg.block[1] * cfg.block[2]
    useful_fma = int(valid.sum()) * nvox_block

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
    total_ms_max, blocks_all = reduce_over_ranks(total_ms, float(n) * args.steps, world, dev, dist)
    value = blocks_all / (total_ms_max * 1e-3)

    # ---- end-to-end leg: the same step through the host-buffer C-ABI call, copies inside the timed region
    e2e_steps = args.e2e_steps if args.e2e_steps is not None else max(3, min(args.steps, 30))
    fixed_p = be.pin(torch.from_numpy(fixed_h))
    moving_p = be.pin(torch.from_numpy(moving_h))
    mask_p = be.pin(torch.from_numpy(mask_h)) if mask_h is not None else None
    ob = be.pin(torch.empty((cap, 3), dtype=torch.int32))
    od = be.pin(torch.empty((cap, 3), dtype=torch.int32))
    on = be.pin(torch.empty((cap,), dtype=torch.float32))
    for _ in range(3):
        nrr.nrr_bm_register_host(fixed_p, moving_p, cfg.block, cfg.stride, cfg.window, cfg.frac, mask_p, ob, od, on)
    barrier()
    e2e_t = 0.0
    for _ in range(e2e_steps):
        flush.zero_()
        be.sync()
        t0 = time.perf_counter()
        rb, rd, rs = nrr.nrr_bm_register_host(fixed_p, moving_p, cfg.block, cfg.stride, cfg.window, cfg.frac, mask_p, ob, od, on)
        e2e_t += time.perf_counter() - t0
    barrier()
    e2e_t_max, e2e_blocks = reduce_over_ranks(e2e_t, float(len(rb)) * e2e_steps, world, dev, dist)
    e2e_value = e2e_blocks / e2e_t_max
    assert np.array_equal(rd.numpy(), disp.cpu().numpy()), "host and device forms disagree"
    h2d = fixed_h.nbytes + moving_h.nbytes + (mask_h.nbytes if mask_h is not None else 0)
    d2h = int(len(rb)) * (12 + 12 + 4) + 4

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (matching): useful FMAs / its own average launch duration
    match_ms = prof["match_ms"] / max(1, prof["match_calls"])
    achieved_tflops = 2.0 * useful_fma / (match_ms * 1e-3) / 1e12
    peak_measured = None
    try:
        peak_measured = nrr.nrr_bm_fp32_peak()
    except Exception as e:  # pragma: no cover
        print("fp32 peak microbenchmark failed: %s" % e, file=sys.stderr)
    info = nrr.nrr_bm_match_info(cfg.dims, cfg.block, cfg.window)
    kernel_name = {2: "match_pair_kernel", 1: "match_rows_kernel", 0: "match_generic_kernel"}[info["kernel"]]
    roofline = {
        "bound": "alu", "kernel": kernel_name, "launch": {"threads": info["threads"], "smem_bytes": info["smem_bytes"],
                                                          "blocks_per_cta": info["blocks_per_cta"], "tma": info["tma"]},
        "achieved": achieved_tflops, "peak": FP32_PEAK_TFLOPS,
        "unit": "TFLOP/s", "frac": achieved_tflops / FP32_PEAK_TFLOPS,
        "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (MEASURED_PEAKS.json has no FP32 figure)",
        "peak_measured_ffma": peak_measured,
        "frac_of_measured_ffma": (achieved_tflops / peak_measured) if peak_measured else None,
        "traffic": None, "useful_fma_per_launch": useful_fma, "kernel_ms": match_ms,
    }

    # ---- the oracle, as it stands, on this box's host cores (a reported baseline, not the target)
    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        import oracle
        r = oracle_step(oracle, cfg, fixed_h, moving_h, mask_h, 32)          # page in, spin up the threads
        rate = r["n_sample"] / max(r["t_match"], 1e-6)
        sample = int(max(64, min(r["n"], rate * 15.0)))                       # ~15 s of CPU work
        r = oracle_step(oracle, cfg, fixed_h, moving_h, mask_h, sample)
        est_step = r["t_select"] + r["t_match"] * (r["n"] / r["n_sample"])
        cpu_baseline = {
            "value": r["n"] / est_step, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
            "sample": "full selection (%.3f s) + matching of %d of %d evenly spaced selected blocks (%.2f s), "
                      "scaled to the whole step" % (r["t_select"], r["n_sample"], r["n"], r["t_match"]),
            "cand_evals_per_sec": r["evals"] / r["t_match"],
        }

    ms_per_step = total_ms_max / args.steps
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "dims": list(cfg.dims), "block": list(cfg.block),
                   "stride": list(cfg.stride), "window": list(cfg.window), "frac": cfg.frac,
                   "blocks_per_pair": int(n), "candidates_per_block": cfg.n_candidates,
                   "l2": "flushed between steps (256 MB write)", "parallelism": "independent pairs per GPU"},
        "cand_evals_per_sec": float(valid.sum()) * args.steps * world / (total_ms_max * 1e-3),
        "ms_per_volume_pair": ms_per_step,
        "phase_ms": {"select": prof["select_ms"] / max(1, prof["select_calls"]),
                     "moving_stats": prof["moving_stats_ms"] / max(1, prof["moving_stats_calls"]),
                     "fixed_records": prof["prep_ms"] / max(1, prof["prep_calls"]),
                     "match": match_ms},
        "match_only": {"blocks_per_sec": n / (match_ms * 1e-3), "cand_evals_per_sec": float(valid.sum()) / (match_ms * 1e-3)},
        "fp32_peak_frac": achieved_tflops / FP32_PEAK_TFLOPS,
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "ms_per_step": 1e3 * e2e_t_max / e2e_steps},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
