"""Multi-GPU sharding of the apply: contiguous alpha-row slabs per rank (every target
amplitude is computed independently), one process per GPU.

Each rank holds the whole input vector (gathers reach any row), computes its slab with bs_apply_rows and
the slabs are exchanged with one all-gather (NCCL on GPUs; the tests drive the same code with gloo on CPU
tensors and a stand-in compute function).  <psi|H|psi> is the all-reduce of the per-slab dots.
bench.py's headline mode runs N independent state vectors (weak scaling, no collective); `bench.py --sharded`
times this module: one state vector, row slabs over the ranks, NCCL all-gather, per-phase device times.

What does not shrink with the number of ranks: every rank transposes the WHOLE input vector for
the beta-only groups (k_transpose, 32 dim bytes per rank per apply) and receives the whole result (16 dim bytes);
the slab kernels themselves scale with the slab.
"""
from __future__ import annotations

from typing import Callable, List, Tuple


def row_slabs(n_rows: int, world: int) -> List[Tuple[int, int]]:
    """Balanced contiguous split of [0, n_rows) into `world` slabs (first n_rows % world slabs are one longer)."""
    base, extra = divmod(n_rows, world)
    out, lo = [], 0
    for r in range(world):
        hi = lo + base + (1 if r < extra else 0)
        out.append((lo, hi))
        lo = hi
    return out


def sharded_apply(apply_rows: Callable, psi_in, psi_out, n_rows: int, row_len: int, group=None, marks=None):
    """psi_out <- H psi_in with every rank computing one slab and all-gathering the rest.

    apply_rows(psi_in, psi_out, row_lo, row_hi) must write psi_out[row_lo*row_len : row_hi*row_len] only
    (bs_apply_rows with op/sector bound).  psi_in must be identical on all ranks.  marks: optional callable invoked
    with "start", "computed", "gathered" on the launching stream (bench.py records CUDA events there).
    """
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    slabs = row_slabs(n_rows, world)
    lo, hi = slabs[rank]
    if marks:
        marks("start")
    apply_rows(psi_in, psi_out, lo, hi)
    if marks:
        marks("computed")
    pieces = [psi_out[a * row_len:b * row_len] for a, b in slabs]
    if all(p.numel() == pieces[0].numel() for p in pieces):
        dist.all_gather(pieces, pieces[rank].clone(), group=group)
    else:  # ragged slabs: one broadcast per slab
        for r, p in enumerate(pieces):
            if p.numel():
                dist.broadcast(p, src=dist.get_global_rank(group, r) if group is not None else r, group=group)
    if marks:
        marks("gathered")
    return psi_out


def sharded_expect(apply_rows: Callable, psi, scratch, n_rows: int, row_len: int, group=None) -> complex:
    """<psi|H|psi> as the all-reduced sum of the per-slab dots (scratch: a vector like psi)."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    lo, hi = row_slabs(n_rows, world)[rank]
    apply_rows(psi, scratch, lo, hi)
    s = slice(lo * row_len, hi * row_len)
    part = torch.vdot(psi[s], scratch[s]).reshape(1)
    part = torch.view_as_real(part).clone()
    dist.all_reduce(part, group=group)
    return complex(part[0, 0].item(), part[0, 1].item())
