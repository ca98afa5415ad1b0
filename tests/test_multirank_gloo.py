"""The N > 1 path of bench.py on CPU: world_size 2, gloo backend, rendezvous on 127.0.0.1.

The FDAS path shards by spectrum with no exchange step: every rank runs the same
plan on its own seeded spectra and the only cross-rank operation is the MAX reduction of the device time.
This test runs exactly those host-side pieces of bench.py in two processes."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        class A:  # the argparse namespace bench.make_workload reads
            config, pair = 1, 0
        wl = bench.make_workload(A, rank)
        my_ms = 2.0 + 3.0 * rank                       # rank 1 is the slow one
        worst = bench.max_over_ranks(my_ms, world)      # CPU tensor -> gloo
        value = bench.whole_job_value(wl.points, world, 4, worst)
        # every rank also learns a checksum of the others' inputs to prove the shards differ
        chk = torch.tensor([float(np.abs(wl.spectrum).sum())], dtype=torch.float64)
        both = [torch.zeros_like(chk) for _ in range(world)]
        dist.all_gather(both, chk)
        out[rank] = (worst, value, wl.points, [float(b.item()) for b in both], wl.spectrum.shape)
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_by_spectrum_and_reduce_time_by_max():
    world = 2
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for r in (0, 1):
        worst, value, points, sums, shape = res[r]
        assert worst == 5.0                                         # MAX over ranks, on every rank
        assert points == 33 * (1 << 16) and shape == (1, 1 << 16)   # same per-rank workload: weak scaling
        assert value == world * points * 4 / 5.0e-3
        assert abs(sums[0] - sums[1]) > 1.0                         # different seeded spectra per rank
    assert res[0][3] == res[1][3]


def test_bench_launches_its_own_ranks():
    """`python bench.py --gpus 2` with no launcher around it starts two ranks itself (torch.distributed.run on
    127.0.0.1) -- here on the CPU-only --dry-run path (gloo), which shares the launcher, the rendezvous and the
    MAX-over-ranks reduction with the GPU path."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run", "--steps", "4", "--config", "1"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout                      # rank 0 alone prints
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["dry_run"] is True
    assert out["ms_per_step"] == 2.0                      # MAX over ranks of (1 + rank) ms
    assert out["value"] == 2 * 33 * (1 << 16) * 4 / (2.0e-3 * 4)
