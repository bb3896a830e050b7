"""Host-side sharding plumbing (paper_2105_04006_b200/sharding.py), covered on CPU with
world_size-2 gloo: object partition of a batch (no collective on the data path), the gather of per-rank best periods,
and the (power, GLOBAL index) all-gather that a frequency-sharded object needs before the library's lsp_best_merge picks
the winner.  The per-rank "periodograms" here come from the CPU oracle and the merge rule is restated in this file
(test infrastructure): what is under test is the partitioning and the gathers, not a kernel.  The CUDA library on
shards -- including lsp_best_merge itself -- is covered by tests/test_gpu_parity.py (-m gpu).
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2105_04006_b200 import sharding
from workloads import make_config


def test_partition_objects_covers_and_balances():
    w = make_config(3, n_obj=200, n_freq=16)
    for world in (1, 2, 3, 8):
        ranges = sharding.partition_objects(w.offsets, world)
        assert len(ranges) == world
        assert ranges[0][0] == 0 and ranges[-1][1] == w.n_obj
        for (a0, a1), (b0, b1) in zip(ranges, ranges[1:]):
            assert a1 == b0 and a0 <= a1
        loads = [int(w.offsets[o1] - w.offsets[o0]) for o0, o1 in ranges]
        assert sum(loads) == w.n_obs
        # a contiguous cut can miss the ideal share by at most one object (<= 500 observations in config 3)
        assert max(abs(x - w.n_obs / world) for x in loads) <= 500


def test_partition_objects_edge_cases():
    assert sharding.partition_objects(np.array([0]), 2) == [(0, 0), (0, 0)]                  # no objects
    assert sharding.partition_objects(np.array([0, 0, 0, 0]), 2) == [(0, 1), (1, 3)]           # all empty: by count
    r = sharding.partition_objects(np.array([0, 10]), 4)                                       # world > n_obj
    assert r[0][0] == 0 and r[-1][1] == 1 and sum(b - a for a, b in r) == 1
    with pytest.raises(ValueError):
        sharding.partition_objects(np.array([0, 5, 3]), 2)
    with pytest.raises(ValueError):
        sharding.partition_objects(np.array([1, 5]), 2)


def test_slice_csr_rebases_offsets():
    w = make_config(3, n_obj=10, n_freq=16)
    off, t, y = sharding.slice_csr(w.offsets, w.t, w.y, 3, 7)
    assert off[0] == 0 and off.size == 5 and off[-1] == t.size == y.size
    assert np.array_equal(np.diff(off), np.diff(w.offsets[3:8]))
    assert np.array_equal(t, w.t[w.offsets[3]:w.offsets[7]])


def test_partition_frequencies_reproduces_the_grid():
    f_min, f_max, n_freq = 0.05, 50.0, 1_000_003
    df = (f_max - f_min) / n_freq
    for world in (1, 2, 3, 8):
        parts = sharding.partition_frequencies(f_min, f_max, n_freq, world)
        assert parts[0][0] == 0 and parts[-1][1] == n_freq
        for (k0, k1, fa, fb), nxt in zip(parts, parts[1:] + [None]):
            assert k1 > k0
            if nxt is not None:
                assert nxt[0] == k1
            # the slice's own spacing and its frequencies equal the global grid's (to FP64 rounding)
            assert abs((fb - fa) / (k1 - k0) - df) <= 1e-15 * f_max
            for i in (0, (k1 - k0) // 2, k1 - k0 - 1):
                assert abs((fa + i * (fb - fa) / (k1 - k0)) - (f_min + (k0 + i) * df)) <= 4e-15 * f_max


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, mode: str, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        oracle.build()
        if mode == "objects":
            # batch sharded by object: each rank evaluates its own CSR slice; rows must equal the unsharded run
            w = make_config(3, n_obj=12, n_freq=300)
            o0, o1 = sharding.partition_objects(w.offsets, world)[rank]
            off, t, y = sharding.slice_csr(w.offsets, w.t, w.y, o0, o1)
            P = oracle.periodogram(off, t, y, w.f_min, w.f_max, w.n_freq)
            idx, pw, per = oracle.best(off, P, w.f_min, w.f_max, w.n_freq)
            counts = [b - a for a, b in sharding.partition_objects(w.offsets, world)]
            allb = sharding.gather_objects((torch.from_numpy(per), torch.from_numpy(pw), torch.from_numpy(idx)), counts)
            q.put((rank, o0, o1, P, tuple(x.numpy() for x in allb)))
        else:
            # one object sharded by frequency range + the best-period max-reduce, with a planted exact tie across ranks
            w = make_config(1)
            k0, k1, fa, fb = sharding.partition_frequencies(w.f_min, w.f_max, w.n_freq, world)[rank]
            P = oracle.periodogram(w.offsets, w.t, w.y, fa, fb, k1 - k0)
            idx, pw, _ = oracle.best(w.offsets, P, fa, fb, k1 - k0)
            power = torch.tensor([pw[0], 7.0, float("nan") if rank == 0 else 1.0, 0.0], dtype=torch.float64)
            index = torch.tensor([idx[0], 5, 3, -1], dtype=torch.int64)
            pp, pk = sharding.gather_best(power, index, k0)
            per, bp, bk = _merge_rule_a7(pp.numpy(), pk.numpy(), w.f_min, w.f_max, w.n_freq)
            q.put((rank, k0, P, per, bp, bk))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def _merge_rule_a7(part_power, part_index, f_min, f_max, n_freq):
    """DESIGN.md reading a7 written out for the test: largest power wins, lowest GLOBAL index on exact ties, NaN / -1 never."""
    n_obj = part_power.shape[1]
    per, bp, bk = np.full(n_obj, np.nan), np.zeros(n_obj), np.full(n_obj, -1, dtype=np.int64)
    for o in range(n_obj):
        cands = [(part_power[r, o], part_index[r, o]) for r in range(part_power.shape[0])
                 if part_index[r, o] >= 0 and not np.isnan(part_power[r, o])]
        if cands:
            p, k = sorted(cands, key=lambda c: (-c[0], c[1]))[0]
            per[o], bp[o], bk[o] = 1.0 / (f_min + k * (f_max - f_min) / n_freq), p, k
    return per, bp, bk


def _run(mode: str, world: int = 2):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, mode, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    return sorted(out, key=lambda x: x[0])


@pytest.mark.timeout(300)
def test_object_sharded_batch_gloo_world2(oracle):
    w = make_config(3, n_obj=12, n_freq=300)
    P_all = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq)
    ridx, rpw, rper = oracle.best(w.offsets, P_all, w.f_min, w.f_max, w.n_freq)
    rows = 0
    for rank, o0, o1, P, allb in _run("objects"):
        assert np.array_equal(P, P_all[o0:o1])          # same arithmetic on the same rows: bit-identical
        rows += o1 - o0
        # every rank ends with the whole batch's best periods, in object order
        assert np.array_equal(allb[2], ridx) and np.array_equal(allb[1], rpw) and np.array_equal(allb[0], rper)
    assert rows == w.n_obj


@pytest.mark.timeout(300)
def test_frequency_sharded_best_period_reduce_gloo_world2(oracle):
    w = make_config(1)
    P_all = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq)
    ridx, rpw, rper = oracle.best(w.offsets, P_all, w.f_min, w.f_max, w.n_freq)
    res = _run("freq")
    P_cat = np.concatenate([r[2] for r in res], axis=1)
    assert np.max(np.abs(P_cat - P_all)) <= 1e-12 * P_all.max()      # slice grids reproduce the global grid
    for rank, k0, P, per, bp, bk in res:
        # object 0: the true best period of config 1, identical on every rank
        assert bk[0] == ridx[0] and abs(bp[0] - rpw[0]) <= 1e-12 * rpw[0] and abs(per[0] - rper[0]) <= 1e-12 * rper[0]
        # object 1: exact tie (7.0) between ranks at local index 5 -> the lower GLOBAL index (rank 0's) wins
        assert bk[1] == 5 and bp[1] == 7.0
        # object 2: rank 0 reports NaN -> never wins; rank 1's (1.0, k0 + 3) does
        assert bk[2] == res[1][1] + 3 and bp[2] == 1.0
        # object 3: no valid frequency on any rank -> index -1, power 0, period NaN
        assert bk[3] == -1 and bp[3] == 0.0 and np.isnan(per[3])
