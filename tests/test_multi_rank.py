"""World-size-2 test of bench.py's multi-GPU bookkeeping on CPU (gloo): the path shards as independent replicas with
no data-path collective; the only exchange is the MAX over ranks of the device time, and the reported
value is the units all ranks processed over that time."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2402_01282_b200 import inputs
    ms_local = [10.0, 14.5][rank]          # this rank's "device time" for 5 steps
    e2e_local = [0.30, 0.20][rank]
    ms, e2e = bench.max_over_ranks([ms_local, e2e_local], world, torch.device("cpu"))
    value = bench.whole_job_value(world, 4, 5, ms)
    # independent signals per replica: different seeds, same recipe
    flm = inputs.flm_real(16, 2 + 1000 * bench.replica_seed_offset(rank), 1)
    digest = torch.tensor([float(np.abs(flm).sum())], dtype=torch.float64)
    both = [torch.zeros_like(digest) for _ in range(world)]
    dist.all_gather(both, digest)
    out.put((rank, ms, e2e, value, [float(b) for b in both]))
    dist.destroy_process_group()


def test_replicas_max_over_ranks_world2():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, e2e, value, digests in res:
        assert ms == 14.5 and e2e == 0.30                      # MAX over ranks, identical on every rank
        assert abs(value - 2 * 4 * 5 / 14.5e-3) < 1e-9          # whole-job units over the slowest rank's time
        assert digests[0] != digests[1]                          # replicas transform different signals


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks([3.0, 1.0], 1, torch.device("cpu")) == [3.0, 1.0]
    assert bench.whole_job_value(1, 4, 10, 50.0) == 4 * 10 / 50e-3


def test_bench_gpus_n_starts_n_ranks():
    """`python bench.py --gpus 2` outside a launcher must itself start 2 ranks (it ran one rank and
    printed n_gpus 1).  --dry-run-cpu: the ranks rendezvous over gloo on 127.0.0.1 and report themselves, no GPU."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR",
                                                           "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "5", "--dry-run-cpu"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2
    ranks = d["ranks"]
    assert sorted(x["rank"] for x in ranks) == [0, 1]
    assert len({x["pid"] for x in ranks}) == 2               # two processes
    assert len({x["seed_offset"] for x in ranks}) == 2       # distinct seeds per replica
    assert d["ms_max"] == 11.0                               # MAX over the ranks' times (10 + rank)
    assert abs(d["value"] - 2 * 4 * 5 / 11.0e-3) < 1e-9


def test_bench_rejects_a_world_size_that_contradicts_gpus():
    import subprocess
    env = dict(os.environ, WORLD_SIZE="3", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run-cpu"],
                       capture_output=True, text=True, timeout=120, env=env)
    assert r.returncode != 0 and "WORLD_SIZE=3" in (r.stderr + r.stdout)
