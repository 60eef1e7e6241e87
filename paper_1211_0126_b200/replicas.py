"""Multi-GPU plumbing: replicas only.

north_star rules out sharding the lattice and halo collectives; the path's independent units
are the noise sources (N_HP + N_LP independent solves).  With N GPUs every
rank holds the whole gauge configuration and works through its own, disjoint, source ids;
there is no data-path collective.  The only exchanges are the barrier and the MAX-over-ranks
of the device-timed region that bench.py's contract asks for (torch.distributed: NCCL on the
GPUs, gloo in the CPU tests).  No arithmetic of the method lives here.
"""
from __future__ import annotations

import os

import numpy as np

REPLICA_STRIDE = 1 << 20   # source ids per rank: rank r owns [r * 2^20, (r + 1) * 2^20)


def replica_source_ids(rank: int, step: int, nrhs: int) -> list:
    """Source ids of batch `step` (0, 1, ...) on rank `rank`: disjoint across ranks and steps."""
    if nrhs < 1 or (step + 1) * nrhs > REPLICA_STRIDE:
        raise ValueError("batch outside this rank's id range")
    base = rank * REPLICA_STRIDE + step * nrhs
    return list(range(base, base + nrhs))


def max_over_ranks(value: float, device=None) -> float:
    """MAX over ranks of a locally measured duration (identity without a process group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_throughput(units_per_rank_per_step: int, steps: int, ms_max: float, world: int) -> float:
    """Units all ranks processed / the slowest rank's time (weak scaling: per-rank work is fixed)."""
    return world * units_per_rank_per_step * steps / (ms_max * 1e-3)


def node_shared_links(wl, local_rank: int, world: int, barrier=None, shm_dir: str = "/dev/shm") -> np.ndarray:
    """The workload's gauge configuration, generated ONCE per node: local rank 0 generates it and writes it to a
    file in shared memory, the other ranks map that file (config 5: 1.2 GB and ~20 s of host work that N ranks
    would otherwise repeat on the same cores).  `barrier` is the job's barrier (None for a single process).
    The file is removed again once every rank holds its mapping; the mapping stays valid."""
    if world == 1 or barrier is None:
        return wl.links()
    job = os.environ.get("TORCHELASTIC_RUN_ID") or os.environ.get("MASTER_PORT", "0")
    path = os.path.join(shm_dir, f"tsm_links_{wl.name}_{wl.gauge_seed}_{job}.npy")
    if local_rank == 0:
        tmp = path + ".tmp"
        with open(tmp, "wb") as f:
            np.save(f, wl.links())
        os.replace(tmp, path)
    barrier()
    U = np.load(path, mmap_mode="r")
    barrier()
    if local_rank == 0:
        os.unlink(path)
    return U
