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


def _worker(rank, world, port, out, shm_dir):
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
        # the gauge configuration is generated once per node and mapped by the other ranks
        from paper_1211_0126_b200 import workloads as W
        wl = W.WORKLOADS[1]
        U = replicas.node_shared_links(wl, rank, world, dist.barrier, shm_dir=shm_dir)
        assert U.shape == (4, wl.V, 3, 3) and bool((U == wl.links()).all())
        dist.barrier()
        assert not [f for f in os.listdir(shm_dir) if f.startswith("tsm_links_")]       # removed again
        if rank == 0:
            out.put((flat[:3], ms, value))
    finally:
        dist.destroy_process_group()


def test_two_replicas_over_gloo(tmp_path):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out, str(tmp_path))) for r in range(2)]
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


def test_gpus_n_without_a_launcher_starts_n_ranks_or_fails_loudly():
    """`python bench.py --gpus 2` with no WORLD_SIZE: the script starts the ranks itself; on a box with fewer than
    2 GPUs it must refuse (non-zero exit, no JSON line) instead of silently timing one replica."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, env=env, timeout=300)
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        assert r.returncode == 0 and '"n_gpus": 2' in r.stdout
    else:
        assert r.returncode != 0 and r.stdout.strip() == "" and "refusing" in r.stderr


def test_reference_arm_lines(monkeypatch, capsys):
    """Both forms of the reference arm's step on a small workload: the LP solve run in full, and the 1-/3-iteration
    sample with the linear extrapolation that config 5 uses; ms_per_step is the time actually spent."""
    import argparse
    import json
    import time
    sys.path.insert(0, ROOT)
    import bench
    from paper_1211_0126_b200 import workloads as W
    args = argparse.Namespace(gpus=1, steps=6, warmup=2, nrhs=0)
    wl = W.WORKLOADS[2]        # 8^3 x 16: a CG iteration is milliseconds, well above timer noise
    for forced in (True, False):
        monkeypatch.setattr(bench, "oracle_runs_in_full", lambda wl, f=forced: f)
        t0 = time.perf_counter()
        bench.run_reference(args, wl)
        wall = time.perf_counter() - t0
        line = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
        assert line["impl"] == "reference" and line["extrapolated"] == (not forced)
        assert line["value"] > 0 and line["cpu_baseline"]["value"] == line["value"] and line["cpu_baseline"]["kind"] == "oracle"
        assert line["ms_per_step"] * 1e-3 * line["steps"] <= wall                      # fits the wall clock
        assert line["config"] == bench.workload_config(wl, 1, 1)           # the same object as our arm's
        if not forced:
            d = line["cpu_baseline"]["detail"]
            assert d["t_per_cg_iteration_s"] > 0 and d["s_per_full_step_extrapolated"] > d["t_3iter_solve_s"]
