"""The N > 1 path of bench.py on CPU: two processes, gloo backend (replicas only).
Checks the host logic that exists for N > 1: disjoint source ids per rank, MAX-over-ranks timing,
whole-job throughput, and that the reference arm runs on rank 0 only."""
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1211_0126_b200 import replicas

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        nrhs, steps = 12, 3
        mine = [i for s in range(steps) for i in replicas.replica_source_ids(rank, s, nrhs)]
        gathered = [None] * world
        dist.all_gather_object(gathered, mine)
        flat = [i for g in gathered for i in g]
        assert len(flat) == world * nrhs * steps and len(set(flat)) == len(flat)      # disjoint across ranks
        local_ms = 100.0 * (1 + rank)                                                  # rank 1 is the slow one
        dist.barrier()
        ms = replicas.max_over_ranks(local_ms)
        assert ms == 100.0 * world
        value = replicas.whole_job_throughput(nrhs, steps, ms, world)
        assert abs(value - world * nrhs * steps / (ms * 1e-3)) < 1e-9
        if rank == 0:
            out.put((flat[:3], ms, value))
    finally:
        dist.destroy_process_group()


def test_two_replicas_over_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    ids, ms, value = out.get(timeout=10)
    assert ids == [0, 1, 2] and ms == 200.0 and abs(value - 2 * 12 * 3 / 0.2) < 1e-9


def test_single_process_is_the_identity():
    assert replicas.max_over_ranks(12.5) == 12.5
    assert replicas.replica_source_ids(3, 2, 4) == [3 * replicas.REPLICA_STRIDE + 8 + k for k in range(4)]
    assert torch.tensor(replicas.whole_job_throughput(12, 3, 1000.0, 1)).item() == 36.0


def test_reference_arm_runs_on_rank_0_only():
    """Under torchrun the other ranks of `bench.py --impl reference` exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "1"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
