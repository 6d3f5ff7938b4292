"""Walker sharding over ranks: walkers are independent units, so
each rank owns a disjoint contiguous range of GLOBAL walker ids and there is no
collective on the data path.  The only communication is the reduction of a few
scalars for reporting (max of the elapsed time, sums of counters), done with
``torch.distributed`` (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import os


def env_rank():
    """(rank, local_rank, world_size) from the torchrun environment (1 process: 0, 0, 1)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def walker_range(rank, world, walkers_per_rank):
    """Weak scaling: rank r owns global walkers [r*Wr, (r+1)*Wr).  The global id is
    what seeds every random stream (workload.rnd64), so a walker's trajectory does
    not depend on how many ranks there are."""
    if not (0 <= rank < world) or walkers_per_rank <= 0:
        raise ValueError("bad shard arguments")
    w0 = rank * walkers_per_rank
    return w0, w0 + walkers_per_rank


def split_walkers(total, world):
    """Strong scaling helper: contiguous ranges covering [0,total), sizes differing by
    at most one (first ``total % world`` ranks take the extra walker)."""
    if total < 0 or world <= 0:
        raise ValueError("bad split arguments")
    base, extra = divmod(total, world)
    out, w0 = [], 0
    for r in range(world):
        w1 = w0 + base + (1 if r < extra else 0)
        out.append((w0, w1))
        w0 = w1
    return out


def reduce_scalars(values, op, device="cpu"):
    """All-reduce a list of python floats with ``op`` in {"max", "sum"}; identity when
    torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return [float(x) for x in t.cpu()]


def barrier():
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
