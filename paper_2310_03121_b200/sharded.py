"""One evaluation sharded over the GPUs of a node by slabs of central atoms (include/aev.h, aev_forward_range;
SURVEY.md 8(e), 8(f) rank 4; the paper's multi-GPU context is PAPER.md:160, 170-177).

One process per GPU, every rank holds the full position array (377 KB at 23.5k atoms: broadcast or all-gathered by
the caller's MD engine), evaluates the AEV rows and the partial forces of its own slab, and the partial forces are
summed with one all-reduce (NCCL over NVLink on GPUs; any torch.distributed backend works, the CPU tests use gloo).
Plumbing only: ranges and collectives; every number is computed by the kernels behind the C ABI.
"""
from __future__ import annotations

from typing import List, Tuple


def central_ranges(n_total: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous (first, count) slabs of the flat atom index, sizes differing by at most one, covering [0, n_total)."""
    if world < 1 or n_total < world:
        raise ValueError("need at least one central atom per rank")
    base, extra = divmod(n_total, world)
    out, first = [], 0
    for r in range(world):
        count = base + (1 if r < extra else 0)
        out.append((first, count))
        first += count
    return out


def sum_partial_forces(partial, dist=None, group=None):
    """In-place sum over the ranks of the partial forces [batch, n_atoms, 3] (all-reduce); returns the tensor."""
    if dist is not None and dist.get_world_size(group) > 1:
        dist.all_reduce(partial, op=dist.ReduceOp.SUM, group=group)
    return partial


def gather_rows(rows, n_total: int, dist=None, group=None):
    """Every rank contributes the rows of its slab (a [count_r, L] tensor, slabs as in central_ranges, rank order);
    returns the full [n_total, L] matrix on every rank (all-gather of unequal slabs by padding to the largest)."""
    import torch
    if dist is None or dist.get_world_size(group) == 1:
        return rows
    world = dist.get_world_size(group)
    ranges = central_ranges(n_total, world)
    most = max(c for _, c in ranges)
    pad = torch.zeros((most, rows.shape[1]), dtype=rows.dtype, device=rows.device)
    pad[: rows.shape[0]] = rows
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([p[:c] for p, (_, c) in zip(parts, ranges)], dim=0)


def forward_backward(ctx, pos, species, box, grad_aev, rank: int, world: int, dist=None, group=None):
    """This rank's share of one aev_forward + aev_backward: returns (aev rows of the slab [count, L] as a view,
    total forces [batch, n_atoms, 3] after the all-reduce).  `ctx` is a paper_2310_03121_b200.Context on this rank's GPU;
    `pos`, `species`, `grad_aev` are the FULL arrays on that GPU (only the slab's rows of grad_aev are read)."""
    n_total = pos.shape[0] * pos.shape[1]
    first, count = central_ranges(n_total, world)[rank]
    aev = ctx.aev_forward_range(pos, species, box, first, count)
    partial = ctx.aev_backward(grad_aev)
    forces = sum_partial_forces(partial, dist, group)
    return aev.view(n_total, -1)[first:first + count], forces
