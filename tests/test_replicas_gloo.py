"""The N>1 path of bench.py on CPU: world_size-2 gloo.  The hot path does not shard (DESIGN.md
8(e): replicas only), so the multi-rank logic is: every rank takes its own disorder realisation,
times are reduced with MAX over ranks, throughput is the sum of the work over the slowest time."""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

import bench  # noqa: E402
import workloads  # noqa: E402


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = workloads.make_workload(2, seed=bench.replica_seed(2, rank))
        local_seconds = 0.010 * (rank + 1)               # rank 1 is the slow one
        slowest = bench.reduce_max(local_seconds, "cpu")
        value = bench.whole_job_gbs(10**9, world, slowest)
        out.put((rank, float(w.params["h"][0]), slowest, value))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_replicas_take_distinct_realisations_and_reduce_with_max():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, h0, t0, v0), (r1, h1, t1, v1) = got
    assert (r0, r1) == (0, 1) and h0 != h1                      # different disorder per rank
    assert t0 == t1 == pytest.approx(0.020)                     # MAX over ranks, same on all ranks
    assert v0 == v1 == pytest.approx(2 * 1e9 / 0.020 / 1e9)     # whole-job aggregate


def test_single_process_helpers_are_identity():
    assert bench.reduce_max(0.5) == 0.5
    assert bench.replica_seed(5, 0) == 1005 and bench.replica_seed(5, 3) == 1305
    n, nnz, s = 10, 40, 4
    c = np.array([0.5, 0.0, 0.25, 0.125])
    full = bench.step_bytes(n, nnz, s)
    assert full == nnz * 12 + 4 * (n + 1) + 8 * s * n * 4
    # K = 3: scaled copy, then k=2 (no Z), k=1 (c_1 == 0: no V), k=0 (full)
    assert bench.pass_bytes(n, nnz, s, c) == 16 * s * n + (full - 8 * s * n) * 2 + full
