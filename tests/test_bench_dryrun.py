"""bench.py end to end on the CPU: main() runs unchanged, with a stand-in backend whose `nrr` adapter forwards the
calls bench.py makes to the emulated library (tests/cuda_emul) and whose events read the host clock.  This checks
the bench's own logic (step, phases, counting of useful FMAs, e2e leg, JSON contract keys) without a GPU; every
number it prints is meaningless as a measurement."""
import io
import json
import time
from contextlib import redirect_stdout

import numpy as np
import pytest
import torch

import _emul
import bench


class _Event:
    def record(self, stream=None):
        self.t = time.perf_counter()

    def elapsed_time(self, other):
        return (other.t - self.t) * 1e3


class _EmulNrr:
    """The subset of the binding bench.py uses, on CPU tensors."""

    NrrError = RuntimeError
    broken_default = False          # test hook: the default kernels give wrong displacements until the fallback is chosen

    def __init__(self):
        self.launches = 0
        self.options = {}

    def nrr_bm_set_option(self, name, value):
        self.options[name] = value
        _emul.set_option(name, value)

    def lib(self):
        return _emul.lib()

    def nrr_bm_register(self, fixed, moving, block, stride, window, frac, mask, capacity, out_blocks, out_n, out_disp, out_ncc):
        b, d, s = _emul.register(fixed.numpy(), moving.numpy(), block, stride, window, frac, None if mask is None else mask.numpy())
        n = min(len(b), capacity)
        out_blocks[:n] = torch.from_numpy(b[:n])
        out_disp[:n] = torch.from_numpy(d[:n])
        if self.broken_default and not self.options.get("force_rows"):
            out_disp[:n, 0] += 1
        out_ncc[:n] = torch.from_numpy(s[:n])
        out_n.fill_(len(b))
        self.launches += 5
        return out_blocks, out_n, out_disp, out_ncc

    def nrr_bm_register_host(self, fixed, moving, block, stride, window, frac, mask, out_blocks, out_disp, out_ncc):
        b, d, s = _emul.register(fixed.numpy(), moving.numpy(), block, stride, window, frac, None if mask is None else mask.numpy())
        k = len(b)
        out_blocks[:k] = torch.from_numpy(b)
        out_disp[:k] = torch.from_numpy(d)
        out_ncc[:k] = torch.from_numpy(s)
        return out_blocks[:k], out_disp[:k], out_ncc[:k]

    def nrr_bm_capacity_bound(self, dims, block, stride, frac):
        return _emul.capacity_bound(dims, block, stride, frac)

    def nrr_bm_plan_create_host(self, fixed, block, stride, window, frac, mask=None):
        return _emul.Plan(fixed.numpy(), block, stride, window, frac, None if mask is None else mask.numpy(), host=True)

    def nrr_bm_plan_create(self, fixed, block, stride, window, frac, mask=None):
        return _emul.Plan(fixed.numpy(), block, stride, window, frac, None if mask is None else mask.numpy(), host=False)

    def nrr_bm_plan_match_host(self, plan, moving, out_disp, out_ncc):
        d, s = plan.match_host(moving.numpy())
        out_disp[:] = torch.from_numpy(d)
        out_ncc[:] = torch.from_numpy(s)
        return out_disp, out_ncc

    def nrr_bm_plan_match_range(self, plan, moving, out_disp, out_ncc, first=0, count=None):
        plan.match(moving.numpy(), first, plan.n - first if count is None else count, out=(out_disp.numpy(), out_ncc.numpy()))
        self.launches += 2
        return out_disp, out_ncc

    def nrr_bm_plan_blocks_host(self, plan):
        return plan.blocks()[0]

    def nrr_bm_plan_destroy(self, plan):
        plan.destroy()

    def nrr_bm_check_async_error(self):
        pass

    def nrr_bm_profile_enable(self, on):
        pass

    def nrr_bm_profile_read(self):
        return {"select_ms": 1.0, "moving_stats_ms": 1.0, "match_ms": 2.0, "prep_ms": 0.5,
                "select_calls": 1, "moving_stats_calls": 1, "match_calls": 1, "prep_calls": 1}

    def nrr_bm_launch_count(self, reset=False):
        v, self.launches = self.launches, 0 if reset else self.launches
        return v

    def nrr_bm_match_info(self, dims, block, window, n=0):
        i = _emul.match_info(dims, block, window)
        return {"fast": bool(i["kernel"]), "kernel": i["kernel"], "threads": i["threads"], "smem_bytes": i["smem_bytes"],
                "tma": bool(i["tma"]), "candidates": i["candidates"], "blocks_per_cta": 0}

    def nrr_bm_fp32_peak(self):
        return 70.0


class _Backend:
    flush_bytes = 1 << 20
    collective_backend = "gloo"

    def __init__(self, local_rank):
        self.nrr = _EmulNrr()
        self.dev = torch.device("cpu")

    def sync(self):
        pass

    def event(self):
        return _Event()

    def stream(self):
        return None

    def pin(self, t):
        return t


def test_bench_main_runs_end_to_end_on_the_emulated_library():
    out = io.StringIO()
    with redirect_stdout(out):
        bench.main(["--workload", "tiny", "--steps", "2", "--warmup", "3", "--e2e-steps", "1", "--no-cpu-baseline"],
                   backend_factory=_Backend)
    line = json.loads(out.getvalue().strip().splitlines()[-1])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks",
                "parity", "ms_per_volume_pair", "phase_ms"):
        assert key in line, key
    par = line["parity"]      # the tiny config against the oracle, outside the timed region
    assert par["ok"] and par["selection_equal"] and par["disp_mismatch_outside_band"] == 0 and par["blocks_checked"] == 259
    assert par["max_abs_dncc"] <= 1e-4 and par["exempt_ties"] >= 0
    assert set(line["ms_per_volume_pair"]) >= {"select", "match", "sum"}
    assert line["e2e"]["plan"]["h2d_bytes_per_step"] == 64 * 64 * 32 * 4 and line["e2e"]["plan"]["value"] > 0
    assert "traffic" in line["roofline"] and "traffic_source" in line["roofline"]
    assert line["metric"] == "blocks_per_sec" and line["unit"] == "blocks/s" and line["steps"] == 2
    assert line["config"]["workload"] == "tiny" and line["config"]["blocks_per_pair"] == 259
    rf = line["roofline"]
    assert rf["bound"] == "alu" and rf["kernel"] == "match_pair_kernel" and rf["unit"] == "TFLOP/s"
    # useful FMAs = sum over blocks of valid candidates x block voxels: at most 259 x 343 x 125, and most of it
    assert 0.7 * 259 * 343 * 125 < rf["useful_fma_per_launch"] <= 259 * 343 * 125
    assert abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    e2e = line["e2e"]
    assert e2e["h2d_bytes_per_step"] == 2 * 64 * 64 * 32 * 4 and e2e["d2h_bytes_per_step"] == 259 * 28 + 4
    assert line["gpu_launches"] == 10 and line["value"] > 0 and e2e["value"] > 0
    assert line["config"]["options"] == {}


def test_bench_option_flag_reaches_the_library_and_the_line():
    """--option NAME=VALUE (the A/B runs of DESIGN.md 6.3): force_rows=1 must time the one-row-per-thread kernel."""
    out = io.StringIO()
    try:
        with redirect_stdout(out):
            bench.main(["--workload", "tiny", "--steps", "1", "--warmup", "3", "--e2e-steps", "1", "--no-cpu-baseline",
                        "--option", "force_rows=1"], backend_factory=_Backend)
    finally:
        _emul.set_option("force_rows", 0)
    line = json.loads(out.getvalue().strip().splitlines()[-1])
    assert line["config"]["options"] == {"force_rows": 1.0}
    assert line["roofline"]["kernel"] == "match_rows_kernel" and line["parity"]["ok"]
    with pytest.raises(SystemExit):
        bench.parse_options(["force_rows"])


def test_reference_arm_times_the_whole_oracle_step_and_agrees_with_cpu_baseline():
    """the reference arm must not under-report the oracle.  On a workload whose whole step fits,
    every reference step IS the whole oracle step; its value and the cpu_baseline leg's value describe the same
    program on the same box and agree (loosely here: two short timings on a shared CPU)."""
    out = io.StringIO()
    with redirect_stdout(out):
        bench.main(["--impl", "reference", "--workload", "tiny", "--steps", "3", "--warmup", "1"])
    ref = json.loads(out.getvalue().strip().splitlines()[-1])
    assert ref["impl"] == "reference" and ref["cpu_baseline"]["kind"] == "oracle" and ref["e2e"]["h2d_bytes_per_step"] == 0
    assert "whole oracle step" in ref["cpu_baseline"]["sample"] and ref["cpu_baseline"]["value"] == ref["value"]
    out = io.StringIO()
    with redirect_stdout(out):
        bench.main(["--workload", "tiny", "--steps", "1", "--warmup", "3", "--e2e-steps", "1", "--no-parity"], backend_factory=_Backend)
    cb = json.loads(out.getvalue().strip().splitlines()[-1])["cpu_baseline"]
    assert cb["cores"] >= 1 and cb["threads_1_value"] > 0 and cb["matching_scaling_1_to_all_threads"] > 0
    assert "whole step" in cb["sample"]
    assert 0.25 < cb["value"] / ref["value"] < 4.0


def test_bench_falls_back_to_the_round_1_kernels_when_parity_fails():
    """Parity is the first gate: wrong results from the default kernels must not be timed.  The run switches, loudly,
    to the kernels measured in round 1 (never to the CPU) and says so in the line."""
    class Broken(_EmulNrr):
        broken_default = True

    class B(_Backend):
        def __init__(self, local_rank):
            super().__init__(local_rank)
            self.nrr = Broken()

    out = io.StringIO()
    try:
        with redirect_stdout(out):
            bench.main(["--workload", "tiny", "--steps", "1", "--warmup", "3", "--e2e-steps", "1", "--no-cpu-baseline"], backend_factory=B)
    finally:
        for name in ("force_rows", "boxstat_generic", "select_generic"):
            _emul.set_option(name, 0)
    line = json.loads(out.getvalue().strip().splitlines()[-1])
    assert line["kernel_fallback"] and "parity" in line["kernel_fallback"]
    assert line["parity"]["ok"] and line["roofline"]["kernel"] == "match_rows_kernel"
