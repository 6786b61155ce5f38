"""Multi-GPU plan of the path: one process per GPU, replicated grid, independent package
streams, ONE sum all-reduce of the per-cell fp64 array.

Packages are independent and the Philox stream is keyed by (seed, frequency, package id), so
the path shards without any data-path exchange until the absorbed field is needed as a whole (by the
temperature update).  Two plans, both host logic only (no arithmetic of the method lives here):

  weak    rank r runs the full package count with seed + r: R independent realisations whose mean is the
          running mean over iterations of reading S12 -- per-GPU work is fixed as R grows.
  strong  rank r runs package ids [r n / R, (r+1) n / R) of the SAME seed: the sum over ranks is the
          single-GPU result up to the order of the fp64 additions.

`combine` is the only collective on the data path: all-reduce(sum) of absorbed_int over the default process group
(NCCL on GPUs, gloo in the CPU tests), then the 1/R of the mean for the weak plan.  `job_totals` is the bookkeeping
of a timed multi-rank run (bench.py): device time = max over ranks, work and launches = sum over ranks.
"""
from __future__ import annotations

from dataclasses import dataclass


@dataclass(frozen=True)
class Shard:
    rank: int
    world: int
    seed: int            # seed this rank simulates with
    pkg_begin: int       # first package id
    pkg_count: int       # number of package ids
    mean_scale: float    # factor applied to the all-reduced sum


def plan(mode: str, rank: int, world: int, n_packages: int, seed: int) -> Shard:
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    if mode == "weak":
        return Shard(rank, world, seed + rank, 0, n_packages, 1.0 / world)
    if mode == "strong":
        b = (rank * n_packages) // world
        e = ((rank + 1) * n_packages) // world
        return Shard(rank, world, seed, b, e - b, 1.0)
    raise ValueError(f"unknown plan {mode!r}")


def combine(absorbed_int, shard: Shard):
    """In-place all-reduce(sum) of the per-cell array (torch tensor, CPU or CUDA) + the plan's scale."""
    import torch.distributed as dist
    if shard.world > 1:
        if not dist.is_initialized():
            raise RuntimeError("torch.distributed is not initialised")
        dist.all_reduce(absorbed_int, op=dist.ReduceOp.SUM)
    if shard.mean_scale != 1.0:
        absorbed_int.mul_(shard.mean_scale)
    return absorbed_int


def init(backend: str, rank: int, world: int, local_rank: int = 0):
    """Join the default process group (rendezvous from MASTER_ADDR / MASTER_PORT in the environment).  backend "nccl":
    the rank is bound to cuda:local_rank first; "gloo": CPU tensors (tests)."""
    import torch
    import torch.distributed as dist
    if world <= 1:
        return
    if backend == "nccl":
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local_rank))
    else:
        dist.init_process_group(backend, rank=rank, world_size=world)


def job_totals(step_ms: float, cell_steps: float, launches: float, world: int, device="cpu") -> dict:
    """Whole-job figures of a timed run: time = MAX over ranks (a step ends when the slowest rank ends), cell-steps and
    kernel launches = SUM over ranks; value = all cell-steps / that time."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(step_ms), float(cell_steps), float(launches)], dtype=torch.float64, device=device)
    if world > 1:
        mx = t.clone()
        dist.all_reduce(mx, op=dist.ReduceOp.MAX)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        t[0] = mx[0]
    ms, steps, n = (float(x) for x in t.tolist())
    return {"step_ms": ms, "cell_steps": steps, "launches": int(round(n)), "value": steps / (ms * 1e-3) if ms > 0 else 0.0}
