"""C-ABI boundary without a GPU: the library loads, exports what include/dd.h declares, validates
arguments, and its host-side delay table equals the oracle's on all five configs.  No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

import dd_workloads as W
import oracle
import paper_1201_5380_b200 as dd

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "dd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dd_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = dd.lib()
    declared = _declared_symbols()
    assert declared == sorted(dd.EXPORTED_SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name


def test_strerror_and_status_codes():
    assert dd.dd_strerror(0) == "success"
    for s in range(-12, 0):
        assert dd.dd_strerror(s) not in ("", "unknown status")
    assert dd.dd_strerror(-99) == "unknown status"


@pytest.mark.parametrize("args", [
    (0, 64e-6, 1500.0, -1.0, 8), (64, 0.0, 1500.0, -1.0, 8), (64, 64e-6, -5.0, -1.0, 8),
    (64, 64e-6, 1500.0, 1.0, 8), (64, 64e-6, 1500.0, 0.0, 8), (64, 64e-6, 1500.0, -1.0, 3),
    (64, 64e-6, 1500.0, -1.0, 16), (2000, 64e-6, 1500.0, -1.0, 8), (64, float("nan"), 1500.0, -1.0, 8),
])
def test_plan_create_rejects_bad_arguments(args):
    with pytest.raises(dd.DDError) as e:
        dd.dd_plan_create(*args)
    assert e.value.status == -2


def test_null_pointers():
    L = dd.lib()
    assert L.dd_plan_create(None, 64, 64e-6, 1500.0, -1.0, 8) == -1
    assert L.dd_plan_destroy(None) == 0
    assert L.dd_set_dm_list(None, None, 1) == -1
    assert L.dd_get_max_delay(None) == -1
    assert L.dd_execute_static(None, 1, None, 16, None, 32, None) == -1


def test_dm_list_validation_leaves_plan_unchanged():
    p = dd.Plan(64, 64e-6, 1500.0, -1.0, 8)
    with pytest.raises(dd.DDError) as e:
        p.set_dm_list([])  # ndm <= 0
    assert e.value.status in (-2,)
    with pytest.raises(dd.DDError) as e:
        dd.dd_get_max_delay(p.handle)
    assert e.value.status == -3
    p.set_dm_list([0.0, 10.0, 20.0])
    before = p.delay_table().copy()
    for bad in ([1.0, -1.0], [float("inf")], [float("nan"), 1.0]):
        with pytest.raises(dd.DDError) as e:
            dd.dd_set_dm_list(p.handle, bad)
        assert e.value.status == -2
    assert np.array_equal(dd.dd_get_delay_table(p.handle, 3, 64), before)
    # a delay that does not fit int32
    with pytest.raises(dd.DDError) as e:
        dd.dd_set_dm_list(p.handle, [1e12])
    assert e.value.status == -7
    assert np.array_equal(dd.dd_get_delay_table(p.handle, 3, 64), before)
    p.close()


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_host_delay_table_equals_oracle(idx):
    cfg = W.CONFIGS[idx]
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(cfg.dm_list())
        tab = p.delay_table()
        ref = oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.dm_list())
        assert tab.dtype == np.int32 and tab.shape == ref.shape
        assert np.array_equal(tab.astype(np.int64), ref)
        assert p.max_delay == int(ref.max())
        info = p.launch_info()
        assert info["smem_bytes"] <= 227 * 1024 and info["n_dm_blocks"] * info["dm_block"] >= cfg.ndm


def test_unsorted_and_repeated_dm_list():
    cfg = W.CONFIGS[2]
    rng = np.random.default_rng(3)
    dms = rng.permutation(np.concatenate([cfg.dm_list()[::40], [0.0, 0.0, 17.25]]))
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(dms)
        assert np.array_equal(p.delay_table().astype(np.int64),
                              oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms))


def test_spread_too_large_for_shared_memory_is_an_error():
    # DM trials 0 and 1e6 in one block: the staged span could never fit on chip
    with dd.Plan(1024, 64e-6, 400.0, -0.05, 8) as p:
        with pytest.raises(dd.DDError) as e:
            p.set_dm_list([0.0, 1.0e6])
        assert e.value.status == -8


def test_execute_argument_checks_need_no_gpu():
    cfg = W.CONFIGS[4]
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        L, h = dd.lib(), p.handle
        assert L.dd_execute(h, 100, 16, 1024, 16, 32, None) == -3          # no DM list
        p.set_dm_list([0.0, 5.0])
        md = p.max_delay
        good_stride = ((100 + md) * 4 // 8 + 15) // 16 * 16
        assert L.dd_execute(h, 100, None, good_stride, 16, 32, None) == -1
        assert L.dd_execute(h, 0, 16, good_stride, 16, 32, None) == -2
        assert L.dd_execute(h, 100, 16, good_stride, 16, 8, None) == -2       # unknown out_nbits
        assert L.dd_execute(h, 100, 16, good_stride + 8, 16, 32, None) == -4  # stride not multiple of 16
        assert L.dd_execute(h, 100, 24, good_stride, 16, 32, None) == -4      # in_ptr not 16-aligned
        assert L.dd_execute(h, 100, 16, good_stride, 18, 32, None) == -4      # out_ptr not element aligned
        assert L.dd_execute(h, 100, 16, 16, 16, 32, None) == -5               # rows too short
        # dd_set_output_stride: bytes between output rows, checked at execute
        assert L.dd_set_output_stride(h, -1) == -2
        assert L.dd_set_output_stride(h, 398) == 0
        assert L.dd_execute(h, 100, 16, good_stride, 16, 32, None) == -4      # not a multiple of the element size
        assert L.dd_set_output_stride(h, 396) == 0
        assert L.dd_execute(h, 100, 16, good_stride, 16, 32, None) == -5      # shorter than a row of 100 float32
        assert L.dd_set_output_stride(h, 0) == 0
    with dd.Plan(8192, 64e-6, 1500.0, -0.01, 4) as p:                        # 8192*15 > 65535
        p.set_dm_list([0.0])
        assert dd.lib().dd_execute(p.handle, 100, 16, 4096, 16, 16, None) == -6
    with dd.Plan(4096, 64e-6, 1500.0, -0.01, 8) as p:
        assert dd.lib().dd_set_batch(p.handle, 0, 0, 0) == -2
        assert dd.lib().dd_set_batch(p.handle, 2, 24, 0) == -4
        assert dd.lib().dd_set_batch(p.handle, 2, 4096 * 64, 1 << 20) == 0


def test_execute_static_argument_checks_need_no_gpu():
    # the argument checks of dd_execute, then DD_ERR_UNSUPPORTED for a plan that does not run the bit-plane kernel --
    # all before the first CUDA call
    cfg = W.CONFIGS[4]
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        L, h = dd.lib(), p.handle
        assert L.dd_execute_static(h, 100, 16, 1024, 16, 32, None) == -3
        p.set_dm_list([0.0, 5.0])
        good_stride = ((100 + p.max_delay) * 4 // 8 + 15) // 16 * 16
        assert L.dd_execute_static(h, 100, None, good_stride, 16, 32, None) == -1
        assert L.dd_execute_static(h, 0, 16, good_stride, 16, 32, None) == -2
        assert L.dd_execute_static(h, 100, 16, good_stride + 8, 16, 32, None) == -4
        assert L.dd_execute_static(h, 100, 24, good_stride, 16, 32, None) == -4
        assert L.dd_execute_static(h, 100, 16, 16, 16, 32, None) == -5
        assert p.launch_info()["variant"] != 3
        assert L.dd_execute_static(h, 100, 16, good_stride, 16, 32, None) == -12
        assert "variant 3" in dd.dd_last_cuda_error()
    assert dd.DD_STATIC_WORKSPACE_BYTES == 64 << 20
    assert "#define DD_STATIC_WORKSPACE_BYTES (64 * 1024 * 1024)" in open(os.path.join(ROOT, "include", "dd.h")).read()


def test_killmask_host_side():
    # the mask changes which channels are summed, not the delay table; NULL removes it
    cfg = W.CONFIGS[2]
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        assert dd.lib().dd_set_killmask(None, None) == -1
        mask = np.ones(cfg.nchans, dtype=np.int32)
        mask[100:300] = 0
        p.set_killmask(mask)                       # before the DM list: remembered
        p.set_dm_list(cfg.dm_list()[:40])
        full = oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.dm_list()[:40])
        assert np.array_equal(p.delay_table().astype(np.int64), full)
        assert p.max_delay == int(full.max())
        p.set_killmask(None)
        p.set_killmask(np.zeros(cfg.nchans, dtype=np.int32))   # every channel killed is legal
        p.set_killmask(mask * 5)
        assert np.array_equal(p.delay_table().astype(np.int64), full)
        with pytest.raises(ValueError):
            p.set_killmask(mask[:10])
    # a mask can bring a plan into the output range: 8192 4-bit channels do not fit uint16, 4000 of them do
    with dd.Plan(8192, 64e-6, 1500.0, -0.01, 4) as p:
        p.set_dm_list([0.0])
        assert dd.lib().dd_execute(p.handle, 100, 16, 4096, 16, 16, None) == -6
        m = np.zeros(8192, dtype=np.int32)
        m[:4000] = 1
        p.set_killmask(m)
        assert p.launch_info()["variant"] in (3, 4)  # 4000 * 15 < 2^16: the bit-plane kernels serve it now
        m[:5000] = 1
        p.set_killmask(m)                           # 5000 * 15 > 65535: still out of range
        assert dd.lib().dd_execute(p.handle, 100, 16, 4096, 16, 16, None) == -6


def test_subband_host_side():
    # argument checks and tables of the sub-band method, no device needed
    cfg = W.CONFIGS[2]
    dms = cfg.dm_list()[:100]
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        L, h = dd.lib(), p.handle
        assert L.dd_set_subband(None, 32, 32) == -1
        assert L.dd_set_subband(h, 33, 32) == -2           # does not divide nchans
        assert L.dd_set_subband(h, 32, 20) == -2           # not a multiple of 16
        assert L.dd_set_subband(h, 128, 32) == -6          # 128 * 3 > 255: intermediate series do not fit 8 bits
        assert L.dd_get_subband_extent(h) == -3            # no DM list
        p.set_subband(32, 32)                              # before the DM list: remembered
        p.set_dm_list(dms)
        nominal, d1, d2 = p.subband_tables()
        rn, r1, r2 = oracle.subband_tables(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms, 32, 32)
        assert np.array_equal(nominal, rn) and np.array_equal(d1, r1) and np.array_equal(d2, r2)
        assert p.subband_extent == oracle.subband_required_samples(1000, r1, r2, 32) - 1000
        # the direct delay table is untouched, and rows shorter than nsamps + extent are refused
        assert np.array_equal(p.delay_table().astype(np.int64),
                              oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms))
        ext = max(p.subband_extent, p.max_delay)
        short = ((100 + ext) * 2 // 8) // 16 * 16          # 2-bit rows a few samples short of nsamps + extent
        assert L.dd_execute_host(h, 100, 16, short, 16, 32) == -5
        assert L.dd_execute(h, 100, 16, short, 16, 32, None) == -5
        p.set_subband(0, 0)
        assert L.dd_get_subband_extent(h) == -2


def test_time_scrunch_argument_checks_need_no_gpu():
    L = dd.lib()
    ok = (4, 1000, 16, 512, 2, 32, 512, 4, None)
    def call(**kw):
        names = ("nrows", "nsamps_out", "in_ptr", "in_stride", "nbits_in", "out_ptr", "out_stride", "nbits_out", "stream")
        a = dict(zip(names, ok))
        a.update(kw)
        return L.dd_time_scrunch(*[a[n] for n in names])
    assert call(in_ptr=None) == -1 and call(out_ptr=None) == -1
    assert call(nrows=0) == -2 and call(nsamps_out=0) == -2 and call(nbits_in=3) == -2 and call(nbits_out=16) == -2
    assert call(nbits_in=2, nbits_out=2) == -6 and call(nbits_in=4, nbits_out=4) == -6 and call(nbits_in=8, nbits_out=8) == -6
    assert call(in_ptr=24) == -4 and call(out_ptr=8) == -4 and call(in_stride=520) == -4 and call(out_stride=500) == -4
    assert call(out_stride=496) == -5          # 1000 4-bit samples = 500 bytes -> 512
    assert call(in_stride=496) == -5           # 512 output bytes of 4-bit sums need 512 input bytes of 2-bit samples


def test_scrunch_set_host_side():
    # dd_scrunch_*: levels, factors and delays equal the oracle's readings T1-T4; argument errors; no GPU needed
    cfg = W.CONFIGS[2]
    dms = cfg.dm_list()
    with dd.ScrunchSet(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, dms, 64) as s:
        lv = s.levels
        diag = oracle.diagonal_dm_np(cfg.nchans, cfg.dt, cfg.f_top, cfg.df)
        fac = oracle.scrunch_factors_np(dms, diag, 64, 3)
        assert [l["factor"] for l in lv] == sorted(set(int(f) for f in fac)) == [1, 2, 4, 8, 16]
        assert lv[0]["dm_diag_micro"] == round(diag * 1e6)
        for l in lv:
            idx = np.nonzero(fac == l["factor"])[0]
            assert (l["first_dm"], l["ndm"]) == (int(idx[0]), len(idx))
            tab = oracle.delay_table(cfg.nchans, cfg.dt * l["factor"], cfg.f_top, cfg.df, np.asarray(dms)[idx])
            assert l["max_delay"] == int(tab.max())
            assert l["nbits"] == {1: 2, 2: 4, 4: 4, 8: 8, 16: 8}[l["factor"]]
        need = s.required_bytes(1 << 16)
        assert need % 16 == 0
        for l in lv:   # every level's own rows fit into what the input must provide
            assert need * 8 // cfg.nbits >= l["factor"] * ((1 << 16) // l["factor"] + l["max_delay"])
        assert need * 8 // cfg.nbits <= (1 << 16) + 16 * lv[-1]["max_delay"] + 16 * 128 * 4
        with pytest.raises(dd.DDError):
            s.required_bytes(8)                      # fewer samples than the largest factor
    with dd.ScrunchSet(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, dms, 1) as s:
        assert [l["factor"] for l in s.levels] == [1] and s.levels[0]["ndm"] == cfg.ndm
    with dd.ScrunchSet(64, 64e-6, 1500.0, -1.0, 8, [0.0, 500.0, 5000.0], 64) as s:
        assert [l["factor"] for l in s.levels] == [1]                       # 8-bit pair sums do not fit 8 bits
    for bad in (dict(dm=[10.0, 5.0], mf=4), dict(dm=[0.0, 1.0], mf=3), dict(dm=[0.0, 1.0], mf=0), dict(dm=[], mf=2),
                dict(dm=[-1.0], mf=2)):
        with pytest.raises(dd.DDError):
            dd.ScrunchSet(64, 64e-6, 1500.0, -1.0, 2, bad["dm"], bad["mf"])
    with pytest.raises(dd.DDError):
        dd.ScrunchSet(64, 64e-6, 1500.0, +1.0, 2, [0.0], 2)                 # observing parameters are validated too


def test_tuning_and_workspace_knobs_host_side():
    """dd_set_tuning / dd_set_workspace_limit / dd_get_workspace_bytes: argument checks and what the planner makes of the
    knobs, without a device (the library reads no environment variables: these calls are the only launch-geometry knobs)."""
    L = dd.lib()
    assert L.dd_set_tuning(None, dd.DD_TUNE_GROUP_SIZE, 4) == -1
    assert L.dd_set_workspace_limit(None, 0) == -1
    assert L.dd_get_workspace_bytes(None) == -1
    cfg = W.CONFIGS[5]
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        for key, value in ((0, 1), (99, 1), (dd.DD_TUNE_GROUP_SIZE, 3), (dd.DD_TUNE_GROUP_SIZE, -1), (dd.DD_TUNE_PAIR_TILES, -2),
                           (dd.DD_TUNE_HOST_SLAB, -1), (7, 1)):
            assert L.dd_set_tuning(p.handle, key, value) == -2, (key, value)
        assert L.dd_set_workspace_limit(p.handle, -1) == -2
        assert L.dd_set_tuning(p.handle, dd.DD_TUNE_HOST_SLAB, 1 << 16) == 0 and L.dd_set_tuning(p.handle, dd.DD_TUNE_HOST_SLAB, 0) == 0
        assert p.workspace_bytes == 0                       # nothing is allocated before the first dd_execute
        p.set_dm_list(cfg.dm_list())
        info = p.launch_info()
        assert info["variant"] == 6 and info["smem_bytes"] <= 227 * 1024 and info["time_block"] == 3072   # rows of four by default
        p.set_tuning(dd.DD_TUNE_GROUP_SIZE, 2).set_dm_list(cfg.dm_list())
        assert p.launch_info()["variant"] == 6              # pairs serve this plan too
        p.set_tuning(dd.DD_TUNE_GROUP_SIZE, 0)
    # the default choice per config: group rows where the cost model says they pay, the bit-plane kernel for the tiny one
    for idx, want in ((1, 3), (2, 6), (3, 6), (4, 6)):
        c = W.CONFIGS[idx]
        with dd.Plan(c.nchans, c.dt, c.f_top, c.df, c.nbits) as p:
            p.set_dm_list(c.dm_list())
            assert p.launch_info()["variant"] == want, idx
    # a promise about the samples keeps the plan on the plane-skipping bit-plane kernel, also when made after the DM list
    c = W.CONFIGS[5]
    with dd.Plan(c.nchans, c.dt, c.f_top, c.df, c.nbits) as p:
        p.set_dm_list(c.dm_list())
        assert p.launch_info()["variant"] == 6
        p.set_input_max(31)
        assert p.launch_info()["variant"] == 3
        p.set_input_max(0)
        assert p.launch_info()["variant"] == 6
    # every variant can be forced; 2-bit input has no rows of two in variant 6
    c = W.CONFIGS[2].reduced(nsamps=4096, ndm=40)
    for variant in (1, 2, 3, 4, 5, 6):
        with dd.Plan(c.nchans, c.dt, c.f_top, c.df, c.nbits, variant=variant) as p:
            p.set_dm_list(c.dm_list())
            assert p.launch_info()["variant"] == variant
    with dd.Plan(c.nchans, c.dt, c.f_top, c.df, c.nbits, variant=6) as p:
        p.set_tuning(dd.DD_TUNE_GROUP_SIZE, 2)
        with pytest.raises(dd.DDError):
            p.set_dm_list(c.dm_list())


def test_tree_host_side():
    # dd_tree_* without a GPU: argument checks, the delays of the recursion and the stage-2 tables against the oracle
    from oracle.oracle_np import piecewise_tree_required_samples, piecewise_tree_tables, tree_delays_np
    L = dd.lib()
    h = ctypes.c_void_p()
    for args in ((1000, 1000, 2), (1024, 48, 2), (1024, 2048, 2), (8192, 8192, 2), (1000, 64, 2), (1 << 17, 64, 2), (1, 1, 2), (64, 64, 3)):
        assert L.dd_tree_create(ctypes.byref(h), *args) == -2
    assert L.dd_tree_create(ctypes.byref(h), 1024, 512, 8) == 0           # (sums beyond 16 bits: 32-bit lanes)
    assert L.dd_tree_destroy(h) == 0
    assert L.dd_tree_create(None, 64, 64, 2) == -1 and L.dd_tree_destroy(None) == 0
    for n in (2, 4, 8, 32, 128, 1024):
        with dd.Tree(n, n, 2) as t:
            assert np.array_equal(t.delays(), tree_delays_np(n))
            assert t.required_samples(100) == 100 + n - 1
    cfg = W.CONFIGS[2]
    dms = np.linspace(0.0, 30.0, 37)
    for sb in (16, 32, 64, 1024):
        with dd.Tree(cfg.nchans, sb, cfg.nbits) as t:
            assert L.dd_tree_get_tables(t.handle, None, None) == -3          # no DM list yet
            if sb == 1024:
                with pytest.raises(dd.DDError) as e:
                    t.set_dm_list(cfg.dt, cfg.f_top, cfg.df, [1000.0, 2000.0])   # 40 k samples across the band
                assert e.value.status == -6
                continue
            t.set_dm_list(cfg.dt, cfg.f_top, cfg.df, dms)
            dprime, dt2 = t.tables()
            o1, o2 = piecewise_tree_tables(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms, sb)
            assert np.array_equal(dprime, o1) and np.array_equal(dt2, o2)
            assert t.required_samples(5000) == piecewise_tree_required_samples(5000, o1, o2, sb)
            for bad in ([], [-1.0], [float("nan")]):
                assert L.dd_tree_set_dm_list(t.handle, cfg.dt, cfg.f_top, cfg.df,
                                             np.asarray(bad + [0.0], dtype=np.float64).ctypes.data_as(ctypes.c_void_p), len(bad)) == -2
            assert L.dd_tree_set_dm_list(t.handle, cfg.dt, cfg.f_top, 0.4, dms.ctypes.data_as(ctypes.c_void_p), 3) == -2
            assert np.array_equal(t.tables()[0], o1)                          # failures left the tables alone
            # execute: argument checks come before the first CUDA call
            need_bytes = (t.required_samples(5000) * 2 // 8 + 15) // 16 * 16
            assert L.dd_tree_execute(t.handle, 5000, None, need_bytes, 16, 32, None) == -1
            assert L.dd_tree_execute(t.handle, 0, 16, need_bytes, 16, 32, None) == -2
            assert L.dd_tree_execute(t.handle, 5000, 16, need_bytes, 16, 8, None) == -2
            assert L.dd_tree_execute(t.handle, 5000, 24, need_bytes, 16, 32, None) == -4
            assert L.dd_tree_execute(t.handle, 5000, 16, need_bytes - 16, 16, 32, None) == -5
            assert L.dd_tree_set_tuning(t.handle, 1, 7) == -2 and L.dd_tree_set_tuning(t.handle, 3, 5) == -2
            assert L.dd_tree_set_tuning(t.handle, 4, 1) == -2 and L.dd_tree_set_tuning(t.handle, 2, 3) == 0
    # the frequency-padded tree: eq. 25 against the oracle; its trials are fixed (no DM list)
    from oracle.oracle_np import padded_tree_map
    for nchans, f_top, df in ((cfg.nchans, cfg.f_top, cfg.df), (24, 1500.0, -8.0), (100, 1581.8, -4.0), (2, 1000.0, -1e-6)):
        with dd.Tree.padded(nchans, f_top, df, 2) as t:
            pos, npad = padded_tree_map(nchans, f_top, df)
            assert np.array_equal(t.padding, pos) and t.nchans == max(npad, 2)
            assert L.dd_tree_set_dm_list(t.handle, cfg.dt, f_top, df, dms.ctypes.data_as(ctypes.c_void_p), 3) == -12
            assert t.required_samples(10) == 10 + t.nchans - 1
    assert L.dd_tree_create_padded(ctypes.byref(h), 4096, 400.0, -0.0244140625, 2) == -2      # 8192 rows: beyond the largest tree
    assert L.dd_tree_create_padded(ctypes.byref(h), 64, 400.0, 0.1, 2) == -2
    with dd.Tree(8, 8, 2) as t:
        assert L.dd_tree_get_padding(t.handle, None) == -2
    with dd.Tree(1024, 256, 8) as t8:
        big = (1 << 20)
        t8.set_dm_list(cfg.dt, cfg.f_top, cfg.df, [0.0, 1.0])
        assert L.dd_tree_execute(t8.handle, 100, 16, big, 16, 16, None) == -6          # 1024 * 255 does not fit uint16
