"""Host-side sharding of the Lomb-Scargle hot path over ranks (one process per GPU).

Every (object, frequency) power is independent, so the path shards with no exchange step:

* a batch is cut into contiguous object ranges balanced by sum N_t (`partition_objects`); each rank runs the
  library on its own CSR slice (`slice_csr`) and owns those rows / best periods: no data-path collective;
* a single huge object is cut by frequency range (`partition_frequencies`); the full periodogram needs nothing,
  the best period needs one max-reduce of (power, index) per object (`reduce_best`: an all-gather of 16 bytes per
  object per rank, lowest index wins exact ties, NaN never wins -- the library's own rule, DESIGN.md a7).

This module holds plumbing only (integer partitioning and one argmax over ranks); it never evaluates a periodogram
and works with any torch.distributed backend (nccl on GPUs; gloo in the CPU tests).
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


def reduce_best(power: torch.Tensor, index: torch.Tensor, k_offset: int, f_min: float, f_max: float, n_freq: int,
                group=None):
    """Best period over frequency-sharded ranks.  `power[n_obj]` / `index[n_obj]` are this rank's fused-argmax results
    on its own grid slice (index -1 = no valid frequency); `k_offset` is the slice's first global frequency number.
    Returns (period, power, global index) on every rank.  One all-gather of (power, index) per object; the winner is
    the largest power, lowest global index on exact ties, NaN / -1 entries never win."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    gidx = torch.where(index >= 0, index + int(k_offset), torch.full_like(index, -1))
    p64 = power.to(torch.float64)
    p64 = torch.where(torch.isnan(p64) | (gidx < 0), torch.full_like(p64, -float("inf")), p64)
    ps = [torch.empty_like(p64) for _ in range(world)]
    ks = [torch.empty_like(gidx) for _ in range(world)]
    dist.all_gather(ps, p64, group=group)
    dist.all_gather(ks, gidx, group=group)
    P = torch.stack(ps)                          # [world, n_obj]
    K = torch.stack(ks)
    pmax = P.max(dim=0).values
    big = torch.iinfo(torch.int64).max
    cand = torch.where((P == pmax.unsqueeze(0)) & (K >= 0), K, torch.full_like(K, big))
    kbest = cand.min(dim=0).values
    none = kbest == big
    kbest = torch.where(none, torch.full_like(kbest, -1), kbest)
    df = (f_max - f_min) / n_freq
    period = 1.0 / (f_min + kbest.to(torch.float64) * df)
    period = torch.where(none, torch.full_like(period, float("nan")), period)
    pw = torch.where(none, torch.zeros_like(pmax), pmax)
    return period.to(power.dtype), pw.to(power.dtype), kbest
