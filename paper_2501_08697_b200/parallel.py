"""Multi-GPU plumbing: one process per GPU, torch.distributed for the rendezvous, NO data-path collective.

The path shards only at the level of independent units: k-points (BASELINE config 2: 64 of
them, Eq. 32 L507 is per k) and, for a Gamma-point config, replicas of the band block.  Ranks never
exchange wave functions; the only collectives are the barrier around the timed region, a MAX over ranks of the
device-measured time, and (for k-sharding) one gather of the nbands eigenvalues per k-point.

The same functions run under `gloo` on CPU (tests, world_size 2) and under `nccl` on the GPUs (bench.py)."""
from __future__ import annotations

import os


def env_world():
    """(rank, world_size, local_rank) as torchrun exports them; (0, 1, 0) for a plain `python` launch."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend=None):
    """Initialise torch.distributed when WORLD_SIZE > 1 (rendezvous on 127.0.0.1 unless MASTER_ADDR is set)."""
    import torch
    import torch.distributed as dist
    rank, world, local = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend, rank=rank, world_size=world)
    return rank, world, local


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()


def _device():
    import torch
    import torch.distributed as dist
    if dist.is_initialized() and dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def barrier():
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
    if torch.cuda.is_available():
        torch.cuda.synchronize()


def max_over_ranks(values):
    """Element-wise MAX over ranks of a list of floats (times measured on each rank's own device)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=_device())
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def shard_units(n_units, rank, world):
    """Contiguous, balanced share of n_units independent units (k-points) for `rank`: sizes differ by at most 1."""
    base, rem = divmod(n_units, world)
    lo = rank * base + min(rank, rem)
    return list(range(lo, lo + base + (1 if rank < rem else 0)))


def gather_rows(local_rows, n_units, ncols):
    """All ranks contribute {unit index: row of ncols floats}; every rank gets the [n_units][ncols] table
    (the one exchange of a k-sharded run: eigenvalues per k-point).  SUM of disjoint contributions."""
    import torch
    import torch.distributed as dist
    t = torch.zeros((n_units, ncols), dtype=torch.float64, device=_device())
    for u, row in local_rows.items():
        t[u] = torch.as_tensor(row, dtype=torch.float64)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t.cpu().numpy()


def aggregate_throughput(units_per_rank, world, ms_max):
    """Whole-job throughput: units processed by all ranks / the slowest rank's device time."""
    return world * units_per_rank / (ms_max * 1e-3)
