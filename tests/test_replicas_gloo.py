"""world_size-2 `gloo` tests (CPU) of the multi-GPU host logic: replicas only, no data-path collective."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    from paper_2405_02410_b200 import replicas, workloads as wl
    cfg = replicas.rank_config(wl.make_config("modelb_128"), rank)
    ic = wl.initial_conditions(cfg)["phi"]
    times, units = replicas.reduce_timings([10.0 + 5.0 * rank, 1.0 - 0.25 * rank], 100 * (rank + 1))
    q.put((rank, cfg["seed"], float(ic.ravel()[0]), times, units))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, x0, t0, u0), (r1, s1, x1, t1, u1) = got
    assert s1 == s0 + 1 and x0 != x1           # independent realisations
    assert t0 == t1 == [15.0, 1.0]             # max over ranks
    assert u0 == u1 == 300.0                   # units of all ranks


def test_reduce_timings_single_process():
    from paper_2405_02410_b200 import replicas
    assert replicas.reduce_timings([3.0], 7) == ([3.0], 7.0)


def test_reference_arm_under_torchrun_prints_one_line():
    """bench.py --impl reference under torchrun: rank 0 alone runs and prints; the other rank exits 0"""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "modelb_128",
           "--ref-budget", "1"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
