"""N > 1 host logic on the CPU (gloo, world_size 2): blocks are independent units, so every
rank matches its own seeded pair and the only collectives are the MAX over ranks of the time and the SUM of the
blocks (bench.py).  The per-rank work runs on the emulated library (tests/cuda_emul), not on a GPU."""
import json
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, outdir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import dataclasses
    import torch.distributed as dist
    import bench
    import _emul
    from nrr_inputs import CONFIGS, make_pair
    dist.init_process_group("gloo", rank=rank, world_size=world)
    small = dataclasses.replace(CONFIGS["tiny"], dims=(32, 32, 16))
    cfg = bench.rank_config(small, rank)
    fixed, moving, mask = make_pair(cfg)
    blocks, disp, ncc = _emul.register(fixed, moving, cfg.block, cfg.stride, cfg.window, cfg.frac, mask)
    my_ms = 10.0 + 5.0 * rank                                   # rank 1 is the slow one
    t_max, n_all = bench.reduce_over_ranks(my_ms, float(len(blocks)), world, None, dist)
    with open(os.path.join(outdir, "rank%d.json" % rank), "w") as f:
        json.dump({"seed": cfg.seed, "n": int(len(blocks)), "t_max": t_max, "n_all": n_all,
                   "checksum": float(np.asarray(disp, np.int64).sum())}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_pairs_and_reduce(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / ("rank%d.json" % k))) for k in range(2)]
    assert r[0]["seed"] != r[1]["seed"]                          # independent pairs
    assert r[0]["t_max"] == r[1]["t_max"] == 15.0                # MAX over ranks
    assert r[0]["n_all"] == r[1]["n_all"] == r[0]["n"] + r[1]["n"]      # SUM over ranks
    assert r[0]["n"] > 0 and r[1]["n"] > 0


def _shard_worker(rank, world, port, outdir):
    """--shard blocks (both images on every processor, the block list distributed): each rank builds
    the same plan, matches its slice of the canonical block list, and one all-gather of 16 B/block completes it."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import dataclasses
    import torch
    import torch.distributed as dist
    import bench
    import _emul
    from nrr_inputs import CONFIGS, make_pair
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = dataclasses.replace(CONFIGS["tiny"], dims=(40, 32, 24))          # the SAME pair on every rank
    fixed, moving, mask = make_pair(cfg)
    plan = _emul.Plan(fixed, cfg.block, cfg.stride, cfg.window, cfg.frac, mask, host=False)
    n = plan.n
    first, count = bench.shard_range(n, rank, world)
    o_disp = torch.full((n, 3), -99, dtype=torch.int32)
    o_ncc = torch.full((n,), -99.0, dtype=torch.float32)
    plan.match(moving, first, count, out=(o_disp.numpy(), o_ncc.numpy()))
    cmax = max(bench.shard_range(n, r, world)[1] for r in range(world))
    send = torch.zeros((cmax, 4), dtype=torch.int32)
    recv = torch.zeros((world, cmax, 4), dtype=torch.int32)
    bench.exchange_block_results(dist, o_disp, o_ncc, n, rank, world, send, recv)
    whole_d, whole_s = plan.match(moving)                                   # what one rank alone computes
    np.save(os.path.join(outdir, "disp%d.npy" % rank), o_disp.numpy())
    with open(os.path.join(outdir, "shard%d.json" % rank), "w") as f:
        json.dump({"n": n, "first": first, "count": count,
                   "equal": bool(np.array_equal(o_disp.numpy(), whole_d) and np.array_equal(o_ncc.numpy(), whole_s))}, f)
    plan.destroy()
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_one_block_list_and_gather(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_shard_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / ("shard%d.json" % k))) for k in range(2)]
    assert r[0]["n"] == r[1]["n"] > 4
    assert r[0]["first"] == 0 and r[0]["count"] == r[1]["first"] and r[1]["first"] + r[1]["count"] == r[0]["n"]
    assert r[0]["equal"] and r[1]["equal"]                       # gathered result == single-rank result, bit for bit
    assert np.array_equal(np.load(tmp_path / "disp0.npy"), np.load(tmp_path / "disp1.npy"))


def _bench_worker(rank, world, port, outdir, shard):
    """bench.py's own main() under torch.distributed (gloo, 2 ranks) on the emulated library: the whole N > 1 host path --
    rendezvous, per-rank step, the pre-timing parity gate, barriers, MAX/SUM reduction, rank 0's JSON line."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import io
    from contextlib import redirect_stdout
    import bench
    from test_bench_dryrun import _Backend
    out = io.StringIO()
    with redirect_stdout(out):
        bench.main(["--gpus", str(world), "--workload", "tiny", "--steps", "1", "--warmup", "3", "--e2e-steps", "1", "--shard", shard],
                   backend_factory=_Backend)
    with open(os.path.join(outdir, "bench_%s_%d.txt" % (shard, rank)), "w") as f:
        f.write(out.getvalue())


@pytest.mark.parametrize("shard", ["blocks", "pairs"])
def test_bench_main_on_two_ranks(tmp_path, shard):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_bench_worker, args=(2, port, str(tmp_path), shard), nprocs=2, join=True)
    out0 = open(tmp_path / ("bench_%s_0.txt" % shard)).read().strip()
    assert open(tmp_path / ("bench_%s_1.txt" % shard)).read().strip() == ""          # rank 0 alone prints
    line = json.loads(out0.splitlines()[-1])
    assert line["n_gpus"] == 2 and line["value"] > 0 and line["parity"]["ok"] and line["kernel_fallback"] is None
    if shard == "blocks":
        # ONE block list of 259 blocks, split 129 + 130, gathered: parity is checked on the gathered result
        assert line["scaling"] == "strong" and line["config"]["blocks_per_pair"] == 259
        assert line["parity"]["blocks_checked"] == 259 and "all-gather" in line["config"]["parallelism"]
    else:
        assert line["scaling"] == "weak" and line["cpu_baseline"] is None
