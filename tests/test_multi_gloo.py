"""N > 1 host logic on CPU: world_size-2 `gloo` processes.

The path shards with no data-path exchange (one beam set per rank); the only collectives
are the SUM of units and the MAX of the per-rank step time that bench.py reports.  These tests run the
same `paper_1201_5380_b200.multi` functions bench.py uses, under torch.distributed with the gloo backend,
and check that the per-rank inputs are the seeded beams each rank is supposed to own (the oracle is the
per-beam check: rank r's transform of its beam equals the single-process transform of that beam).
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

import dd_workloads as W
import oracle
from paper_1201_5380_b200 import multi


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, nbeams: int, ret):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    assert multi.env_rank() == (rank, rank, world)
    assert multi.init_process_group("gloo")
    multi.barrier()
    mine = multi.shard_beams(nbeams, world, rank)
    # every rank dedisperses (with the oracle: no GPU here) only the beams it owns
    cfg = W.CONFIGS[5].reduced(nsamps=300, ndm=6, nchans=32, nbeams=nbeams)
    tab = oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.dm_list())
    sums = {}
    for b in mine:
        packed, _ = W.gen_packed(cfg, int(tab.max()), beams=[b])
        sums[b] = int(oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab).sum())
    units = len(mine) * cfg.ndm * cfg.nsamps
    ms = 10.0 * (rank + 1)                         # rank 1 is the slow one
    value, max_ms = multi.job_throughput(units, ms)
    total = multi.sum_over_ranks(units)
    # DM slabs (input replicated, rows disjoint) and time slabs (halo of max_delay samples): each rank runs the
    # transform of its slab only; the slabs are then assembled with the optional all_gather and compared
    # with the single-process transform by the parent
    one = W.CONFIGS[2].reduced(nsamps=700, ndm=40, nchans=24)
    tab1 = oracle.delay_table(one.nchans, one.dt, one.f_top, one.df, one.dm_list())
    maxd = int(tab1.max())
    packed1, _ = W.gen_packed(one, maxd)
    rows = packed1[0].numpy()
    lo, hi = multi.shard_dm_slabs(one.ndm, world, rank)
    slab = oracle.dedisperse(rows, one.nbits, one.nsamps, tab1[lo:hi]) if hi > lo else np.zeros((0, one.nsamps), np.int64)
    whole = multi.gather_dm_rows(torch.from_numpy(slab.astype(np.int64)), one.ndm, world)
    t_lo, t_hi, i_lo, i_hi = multi.shard_time_slabs(one.nsamps, world, rank, maxd)
    unp = oracle.unpack(rows, one.nbits, one.nsamps + maxd)[:, i_lo:i_hi]          # this rank's input slab only
    unp = np.pad(unp, ((0, 0), (0, -unp.shape[1] % 4)))                             # whole bytes of 2-bit samples
    tslab = oracle.dedisperse(W.pack_rows(torch.from_numpy(unp.astype(np.uint8)), one.nbits).numpy(), one.nbits,
                              t_hi - t_lo, tab1)
    ret[rank] = dict(mine=mine, sums=sums, value=value, max_ms=max_ms, total=total,
                     mx=multi.max_over_ranks(float(rank)), dm_bounds=(lo, hi), whole=whole.numpy(),
                     t_bounds=(t_lo, t_hi), tslab=np.asarray(tslab))
    multi.barrier()
    torch.distributed.destroy_process_group()


@pytest.mark.timeout(180)
def test_world2_gloo_beam_sharding_and_timing_reduction():
    world, nbeams = 2, 5
    port = _free_port()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, port, nbeams, ret), nprocs=world, join=True)
    r0, r1 = ret[0], ret[1]
    # disjoint, complete, balanced, contiguous
    assert r0["mine"] == [0, 1, 2] and r1["mine"] == [3, 4]
    # whole-job value = all units / slowest rank's time, identical on both ranks
    cfg_units = nbeams * 6 * 300
    assert r0["total"] == r1["total"] == cfg_units
    assert r0["max_ms"] == r1["max_ms"] == 20.0
    assert r0["value"] == r1["value"] == pytest.approx(cfg_units / 20e-3)
    assert r0["mx"] == r1["mx"] == 1.0
    # each rank worked on its own seeded beams: the sums equal a single-process evaluation of those beams
    cfg = W.CONFIGS[5].reduced(nsamps=300, ndm=6, nchans=32, nbeams=nbeams)
    tab = oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.dm_list())
    packed, _ = W.gen_packed(cfg, int(tab.max()))
    for b in range(nbeams):
        want = int(oracle.dedisperse(packed[b].numpy(), cfg.nbits, cfg.nsamps, tab).sum())
        got = (r0["sums"] if b in r0["sums"] else r1["sums"])[b]
        assert got == want
    assert len({r0["sums"][b] for b in r0["sums"]} | {r1["sums"][b] for b in r1["sums"]}) == nbeams


    # DM slabs and time slabs: assembled shards == the single-process transform
    one = W.CONFIGS[2].reduced(nsamps=700, ndm=40, nchans=24)
    tab1 = oracle.delay_table(one.nchans, one.dt, one.f_top, one.df, one.dm_list())
    packed1, _ = W.gen_packed(one, int(tab1.max()))
    ref = oracle.dedisperse(packed1[0].numpy(), one.nbits, one.nsamps, tab1)
    assert r0["dm_bounds"] == (0, 32) and r1["dm_bounds"] == (32, 40)              # 3 DM blocks of 16: 2 + 1 (ragged)
    assert np.array_equal(r0["whole"], ref) and np.array_equal(r1["whole"], ref)
    assert r0["t_bounds"] == (0, 384) and r1["t_bounds"] == (384, 700)
    assert np.array_equal(np.concatenate([r0["tslab"], r1["tslab"]], axis=1), ref)


def test_dm_and_time_slab_properties():
    for n in (0, 1, 15, 16, 17, 1200, 4096):
        for world in (1, 2, 3, 8):
            b = [multi.shard_dm_slabs(n, world, r) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == n and all(b[i][1] == b[i + 1][0] for i in range(world - 1))
            assert all((lo % 16 == 0 or lo == hi == n) and lo <= hi for lo, hi in b)   # empty slabs sit at the end
            sizes = [-(-(hi - lo) // 16) for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1
    for n in (0, 100, 128, 1 << 19, (1 << 19) + 77):
        for world in (1, 2, 4, 8):
            s = [multi.shard_time_slabs(n, world, r, 20476) for r in range(world)]
            assert s[0][0] == 0 and s[-1][1] == n and all(s[i][1] == s[i + 1][0] for i in range(world - 1))
            assert all(t_lo % 128 == 0 or t_lo == t_hi == n for t_lo, t_hi, _, _ in s)
            assert all(i_hi == t_hi + 20476 for t_lo, t_hi, _, i_hi in s if t_hi > t_lo)
    with pytest.raises(ValueError):
        multi.shard_dm_slabs(10, 2, 2)
    with pytest.raises(ValueError):
        multi.shard_time_slabs(10, 2, 0, -1)


def test_shard_beams_properties():
    for nbeams in (0, 1, 5, 13, 16):
        for world in (1, 2, 3, 4, 8):
            parts = [multi.shard_beams(nbeams, world, r) for r in range(world)]
            assert sorted(sum(parts, [])) == list(range(nbeams))
            assert max(map(len, parts)) - min(map(len, parts)) <= 1
    with pytest.raises(ValueError):
        multi.shard_beams(4, 2, 2)


def test_single_process_reductions_are_identity():
    assert multi.max_over_ranks(3.5) == 3.5 and multi.sum_over_ranks(2.0) == 2.0
    v, ms = multi.job_throughput(1000.0, 10.0)
    assert v == pytest.approx(1e5) and ms == 10.0
