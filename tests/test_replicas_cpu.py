"""Multi-process CPU tests (gloo, world_size 2) of the replicas plumbing (the path
shards by instance only, no data-path collective): rank environment, instance ranges, barrier, MAX / SUM
over ranks, and the rank-0-only reference arm of bench.py."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch.multiprocessing as mp

from paper_2601_14414_b200 import replicas, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    r, lr, w = replicas.init("gloo")
    assert (r, lr, w) == (rank, rank, world)
    replicas.barrier()
    mx = replicas.max_over_ranks(10.0 + rank)           # the per-rank device time of the timed region
    sm = replicas.sum_over_ranks(float(rank + 1))
    lo, hi = replicas.weak_instance_range(8, rank)
    slo, shi = replicas.strong_instance_range(11, rank, world)
    # every rank generates ITS OWN instances of the global seeded stream: same data as a single-process slice
    p = wl.config4(batch=hi - lo, first_instance=lo)
    ref = wl.config4(batch=16)
    same = bool(np.array_equal(p.A, ref.A[lo:hi]) and np.array_equal(p.x0, ref.x0[lo:hi]))
    replicas.barrier()
    out.put((rank, mx, sm, lo, hi, slo, shi, same))


def test_world_size_2_gloo_replicas():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [11.0, 11.0]          # MAX over ranks, identical on every rank
    assert [r[2] for r in res] == [3.0, 3.0]
    assert [(r[3], r[4]) for r in res] == [(0, 8), (8, 16)]          # weak scaling: disjoint, fixed per-rank work
    assert [(r[5], r[6]) for r in res] == [(0, 6), (6, 11)]          # strong scaling: balanced cover of 11 instances
    assert all(r[7] for r in res)


def test_instance_ranges_cover_without_overlap():
    for total in (1, 7, 64, 4096):
        for world in (1, 2, 3, 8):
            spans = [replicas.strong_instance_range(total, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == total
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1


def test_reference_arm_prints_on_rank_0_only():
    """bench.py --impl reference under torchrun (N > 1): rank 0 alone runs and prints, the others exit 0."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "solves/s"
