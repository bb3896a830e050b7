"""Host-side sharding of the Lomb-Scargle hot path over ranks (one process per GPU).

Every (object, frequency) power is independent, so the path shards with no exchange step:

* a batch is cut into contiguous object ranges balanced by sum N_t (`partition_objects`); each rank runs the
  library on its own CSR slice (`slice_csr`) and owns those rows / best periods: no data-path collective;
* a single huge object is cut by frequency range (`partition_frequencies`); the full periodogram needs nothing,
  the best period needs one max-reduce of (power, index) per object: `gather_best` all-gathers 16 bytes per object per
  rank and the library's `lsp_best_merge` (include/lsp.h) picks the winner with its own rule (DESIGN.md a7).

This module holds plumbing only (integer partitioning, CSR slicing, all-gathers); it never evaluates a periodogram, an
argmax or a period -- those live behind the C ABI -- and works with any torch.distributed backend (nccl on GPUs; gloo in
the CPU tests).
"""
from __future__ import annotations

from typing import List, Tuple

import numpy as np
import torch


def partition_objects(offsets, world: int) -> List[Tuple[int, int]]:
    """Contiguous object ranges [(o0, o1)] * world with sum N_t as even as a contiguous cut allows: range r ends at
    the first object boundary whose cumulative observation count reaches (r + 1)/world of the total (ties: the
    earlier boundary).  Ranges may be empty (world > n_obj); they always cover [0, n_obj) in order."""
    off = np.asarray(offsets, dtype=np.int64)
    if off.ndim != 1 or off.size < 1 or off[0] != 0 or np.any(np.diff(off) < 0):
        raise ValueError("offsets must be a non-decreasing CSR array starting at 0")
    if world < 1:
        raise ValueError("world must be >= 1")
    n_obj = off.size - 1
    total = int(off[-1])
    bounds = [0]
    for r in range(1, world):
        if total == 0:        # nothing to balance: split by object count
            b = (n_obj * r) // world
        else:
            target = total * r / world
            hi = int(np.searchsorted(off, target, side="left"))      # first boundary with cum >= target
            hi = min(max(hi, 0), n_obj)
            lo = max(hi - 1, 0)
            b = lo if abs(off[lo] - target) <= abs(off[hi] - target) else hi
        bounds.append(max(b, bounds[-1]))
    bounds.append(n_obj)
    return [(bounds[r], bounds[r + 1]) for r in range(world)]


def slice_csr(offsets, t, y, o0: int, o1: int):
    """The CSR batch of objects [o0, o1): (offsets rebased to 0, t slice, y slice).  Views, no copies of t / y."""
    off = np.asarray(offsets, dtype=np.int64)
    a, b = int(off[o0]), int(off[o1])
    return off[o0:o1 + 1] - a, t[a:b], y[a:b]


def partition_frequencies(f_min: float, f_max: float, n_freq: int, world: int):
    """Cut the half-open grid f_k = f_min + k df, df = (f_max - f_min)/n_freq into `world` contiguous
    index ranges.  Returns [(k0, k1, f_min_r, f_max_r)]: rank r runs a plan on (f_min_r, f_max_r, k1 - k0), whose own
    spacing (f_max_r - f_min_r)/(k1 - k0) equals df, so its frequency number i is the global k0 + i."""
    if world < 1 or n_freq < 1:
        raise ValueError("world and n_freq must be >= 1")
    df = (f_max - f_min) / n_freq
    out = []
    for r in range(world):
        k0, k1 = (n_freq * r) // world, (n_freq * (r + 1)) // world
        out.append((k0, k1, f_min + k0 * df, f_min + k1 * df))
    return out


def gather_best(power: torch.Tensor, index: torch.Tensor, k_offset: int, group=None):
    """Frequency-sharded best period, plumbing half: every rank contributes its fused-argmax results on its own grid
    slice (`power[n_obj]`, `index[n_obj]` with -1 = no valid frequency; `k_offset` = the slice's first GLOBAL frequency
    number) and receives the candidates of all ranks as (part_power [world, n_obj], part_index [world, n_obj], GLOBAL
    indices, -1 kept).  One all-gather of 16 bytes per object per rank; no arithmetic on the powers happens here -- the
    winner is picked by the library (`Plan.best_merge` = lsp_best_merge of include/lsp.h: largest power, lowest index on
    exact ties, NaN / -1 never win, period = 1/f_k on the global grid)."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    gidx = torch.where(index >= 0, index + int(k_offset), torch.full_like(index, -1))
    ps = [torch.empty_like(power) for _ in range(world)]
    ks = [torch.empty_like(gidx) for _ in range(world)]
    dist.all_gather(ps, power.contiguous(), group=group)
    dist.all_gather(ks, gidx, group=group)
    return torch.stack(ps), torch.stack(ks)


def gather_objects(best, counts: List[int], group=None):
    """Object-sharded batch, plumbing half: rank r holds (period, power, index) tensors of its own counts[r] objects;
    returns the three arrays of the whole batch, in object order, on every rank (ranges from `partition_objects` are
    contiguous and ordered, so concatenation by rank is the batch order).  No arithmetic."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    assert len(counts) == world
    n_max = max(counts) if counts else 0
    out = []
    for x in best:
        pad = torch.zeros(n_max, dtype=x.dtype, device=x.device)
        pad[:x.numel()] = x
        parts = [torch.empty_like(pad) for _ in range(world)]
        dist.all_gather(parts, pad, group=group)
        out.append(torch.cat([parts[r][:counts[r]] for r in range(world)]))
    return tuple(out)
