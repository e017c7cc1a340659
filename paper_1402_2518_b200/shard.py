"""Host-side sharding of the pixel axis over ranks.

Eq. 2 of the paper is a sum of independent per-pixel terms and the constraints are per
pixel: ranks own disjoint contiguous blocks of pixels, the library is replicated, and
the data path needs no collective.  The only communication is the barrier around the timed region and
the max-over-ranks of the step time (bench.py), plus an optional gather of the outputs.
No solver arithmetic lives here.
"""
from __future__ import annotations

from typing import Tuple


def pixel_block(N: int, rank: int, world: int) -> Tuple[int, int]:
    """Half-open range [lo, hi) of the pixels rank `rank` of `world` owns: contiguous, disjoint, covering
    0..N, sizes differing by at most one (the first N % world ranks take the extra pixel)."""
    if world < 1 or not (0 <= rank < world) or N < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, N >= 0")
    base, extra = divmod(N, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def cube_block(rank: int, cubes_per_rank: int) -> Tuple[int, int]:
    """Weak scaling (bench.py): every rank owns its own `cubes_per_rank` cubes of the synthetic stack."""
    if rank < 0 or cubes_per_rank < 0:
        raise ValueError("need rank >= 0, cubes_per_rank >= 0")
    return rank * cubes_per_rank, (rank + 1) * cubes_per_rank


def launch_plan(gpus: int, environ, visible_devices: int, argv, python: str, port: int):
    """How `bench.py --gpus N` starts its ranks.  Returns ("inline", None) when this process is a rank already
    (WORLD_SIZE set by torchrun) or one GPU is asked for, else ("spawn", cmd): the torchrun command line that starts
    one rank per GPU on this node with the same arguments (rendezvous on 127.0.0.1: the container's hostname may not
    resolve).  Asking for more GPUs than the node shows is an error, never a silent one-rank run."""
    if gpus < 1:
        raise ValueError("--gpus must be >= 1")
    if "WORLD_SIZE" in environ:
        world = int(environ["WORLD_SIZE"])
        if world != gpus:
            raise ValueError(f"--gpus {gpus} but the launcher started WORLD_SIZE={world} ranks")
        return "inline", None
    if gpus == 1:
        return "inline", None
    if visible_devices < gpus:
        raise ValueError(f"--gpus {gpus} but only {visible_devices} CUDA device(s) are visible on this node")
    cmd = [python, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + list(argv)
    return "spawn", cmd


def max_over_ranks(value: float, device=None) -> float:
    """Maximum of a per-rank scalar (step time) over the process group; identity without a group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_blocks(local, N: int, device=None):
    """All-gather of per-rank output blocks (rows = the rank's pixel_block) into the full N-row tensor,
    on every rank.  Blocks may differ in length by one row, so they are padded to the longest."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    world, rank = dist.get_world_size(), dist.get_rank()
    longest = -(-N // world)
    lo, hi = pixel_block(N, rank, world)
    assert local.shape[0] == hi - lo
    pad = torch.zeros((longest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: hi - lo] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    out = []
    for r in range(world):
        a, b = pixel_block(N, r, world)
        out.append(parts[r][: b - a])
    return torch.cat(out, 0)
