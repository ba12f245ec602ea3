"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, bit-exact.

Small cases compare every output element; the full BASELINE.json sizes compare sampled outputs that the
oracle computes one by one (plus whole DM rows for the bench config).  All inputs are seeded and
synthetic (dd_workloads); no expected value comes from the CUDA path.
"""
import numpy as np
import pytest
import torch

import dd_workloads as W
import oracle
import paper_1201_5380_b200 as dd

pytestmark = pytest.mark.gpu

_TORCH_OUT = {"f32": torch.float32, "u32": torch.int32, "u16": torch.int16}
_NP_VIEW = {"f32": np.float32, "u32": np.uint32, "u16": np.uint16}


def _oracle_table(cfg, dms=None):
    return oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.dm_list() if dms is None else dms)


def _gpu_transform(cfg, packed_dev, stride, dms, out_kind=None, nsamps=None, variant=0):
    """Run dd_execute on device-resident packed input [nbeams][nchans][stride]; returns a numpy array
    [nbeams][ndm][nsamps] of the output type."""
    out_kind = out_kind or cfg.out
    nsamps = nsamps or cfg.nsamps
    nbeams = packed_dev.shape[0]
    ndm = len(dms)
    out = torch.full((nbeams, ndm, nsamps), -1, dtype=_TORCH_OUT[out_kind], device="cuda")
    code = {"f32": 32, "u32": -32, "u16": 16}[out_kind]
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=variant) as p:
        p.set_dm_list(dms)
        if nbeams > 1:
            p.set_batch(nbeams, packed_dev.stride(0), out.stride(0) * out.element_size())
        p.execute(nsamps, packed_dev, stride, out, code, torch.cuda.current_stream())
        torch.cuda.synchronize()
        info = p.launch_info()
        assert (info["last_launches"] == {3: 2, 5: 2}.get(info["variant"], 1) or (info["variant"] in (4, 6) and info["last_launches"] >= 3)) \
            and (variant == 0 or info["variant"] == variant)
    return out.cpu().numpy().view(_NP_VIEW[out_kind])


def _full_compare(cfg, dms=None, out_kinds=None, nsamps=None, variant=0):
    dms = cfg.dm_list() if dms is None else np.asarray(dms, dtype=np.float64)
    nsamps = nsamps or cfg.nsamps
    tab = _oracle_table(cfg, dms)
    # pulses follow the config's own DM list (their tracks come from the oracle's table)
    ptab = _oracle_table(cfg)
    pulses = W.make_pulses(cfg, lambda idx: ptab[idx])
    max_delay = int(max(tab.max(), ptab.max() if pulses is not None else 0))
    packed, stride = W.gen_packed(cfg, max_delay, pulses)
    packed_dev = packed.cuda()
    for kind in (out_kinds or [cfg.out]):
        got = _gpu_transform(cfg, packed_dev, stride, dms, kind, nsamps, variant)
        for b in range(cfg.nbeams):
            ref = oracle.cast_out(oracle.dedisperse(packed[b].numpy(), cfg.nbits, nsamps, tab), kind)
            assert got[b].shape == ref.shape
            bad = np.nonzero(got[b] != ref)
            assert bad[0].size == 0, (f"{cfg.name} {kind} beam {b}: {bad[0].size} mismatches, first at "
                                      f"d={bad[0][0]} t={bad[1][0]} got={got[b][bad[0][0], bad[1][0]]} "
                                      f"ref={ref[bad[0][0], bad[1][0]]}")


# ------------------------------------------------------------------ small cases, every element compared
def test_cfg1_full_u32_and_f32():
    _full_compare(W.CONFIGS[1], out_kinds=["u32", "f32", "u16"])


@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4])
def test_cfg2_reduced_several_tiles_ragged_tail(variant):
    # 1024 channels, 2-bit, 70 DMs (3 DM blocks of 32 / 5 of 16, last ragged), 3 time tiles + ragged tail of 77 samples
    _full_compare(W.CONFIGS[2].reduced(nsamps=3 * 1280 + 77, ndm=70), variant=variant)


def test_variant3_bitplane_tiles_and_channel_padding():
    # bit-plane kernel: 5120-sample tiles (2 tiles + ragged tail), 16-DM blocks (ragged), channel counts around
    # the 32-channel stage (padded with zero channels) and the ring depth
    _full_compare(W.CONFIGS[2].reduced(nsamps=2 * 5120 + 333, ndm=37), out_kinds=["f32", "u32", "u16"], variant=3)
    for nchans in (1, 31, 32, 33, 64, 65, 95, 129, 1023, 1365):
        _full_compare(W.CONFIGS[2].reduced(nsamps=1283, ndm=3, nchans=nchans), out_kinds=["u32"], variant=3)


def test_variant3_extreme_values_fill_all_planes():
    # all samples 3 with 1365 channels: every sum is 4095 = 2^12 - 1 (all twelve planes set); all samples 0
    cfg = W.CONFIGS[2].reduced(nsamps=700, ndm=5, nchans=1365)
    tab = _oracle_table(cfg)
    nbytes = (cfg.nsamps + int(tab.max()) + 3) // 4
    stride = (nbytes + 15) // 16 * 16
    for fill, want in ((0xFF, 4095), (0x00, 0)):
        packed = torch.full((1, cfg.nchans, stride), fill, dtype=torch.uint8)
        got = _gpu_transform(cfg, packed.cuda(), stride, cfg.dm_list(), "u32", cfg.nsamps, 3)
        ref = oracle.dedisperse(packed[0].numpy(), 2, cfg.nsamps, tab)
        assert np.array_equal(got[0], ref) and int(ref.max()) == want and int(ref.min()) == want


@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_variant4_pair_rows(nbits):
    # pair rows: one pre-summed row per (channel pair, delay difference), every trial adds the row of its own
    # difference -- exact.  Channel counts around the stage size (16 / 8 pairs), odd counts (a last single channel),
    # several tiles with a ragged tail, all output types, unsorted DM list, two beams through device and host paths
    full = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]]

    class base:   # reduced copies of the config with one beam unless asked otherwise
        @staticmethod
        def reduced(**kw):
            kw.setdefault("nbeams", 1)
            return full.reduced(**kw)

    _full_compare(base.reduced(nsamps=2 * 3072 + 333, ndm=37, nchans=200), out_kinds=["f32", "u32", "u16"], variant=4)
    for nchans in (1, 2, 3, 15, 16, 17, 31, 33, 63, 65, 257):
        _full_compare(base.reduced(nsamps=1283, ndm=3, nchans=nchans), out_kinds=["u32"], variant=4)
    cfg = base.reduced(nsamps=1000, ndm=24, nchans=96)
    dms = np.asarray(cfg.dm_list())[np.random.default_rng(4).permutation(cfg.ndm)]
    _full_compare(cfg, dms=dms, out_kinds=["u32"], variant=4)
    cfg = base.reduced(nsamps=3072 + 500, ndm=19, nchans=70, nbeams=2)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    dev = packed.cuda()
    mask = (np.arange(cfg.nchans) % 4 != 1).astype(np.int32)
    out = torch.full((2, cfg.ndm, cfg.nsamps), -1, dtype=torch.float32, device="cuda")
    h_out = torch.zeros((2, cfg.ndm, cfg.nsamps), dtype=torch.float32).pin_memory()
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=4) as p:
        p.set_killmask(mask)
        p.set_dm_list(cfg.dm_list())
        assert p.launch_info()["variant"] == 4
        p.set_batch(2, dev.stride(0), out.stride(0) * 4)
        p.execute(cfg.nsamps, dev, stride, out, 32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        p.execute_host(cfg.nsamps, packed.contiguous().pin_memory(), stride, h_out, 32)
    for b in range(2):
        ref = oracle.dedisperse(packed[b].numpy(), cfg.nbits, cfg.nsamps, tab, mask=mask).astype(np.float32)
        assert np.array_equal(out[b].cpu().numpy(), ref) and np.array_equal(h_out[b].numpy(), ref)


@pytest.mark.parametrize("nbeams", [1, 2])
@pytest.mark.parametrize("tiles_per_group", [1, 2, 3])
@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_variant4_time_axis_split_into_groups(nbits, tiles_per_group, nbeams):
    # The pair-row launcher builds and transforms the rows per GROUP of time tiles (two buffers and two internal
    # streams that alternate); with the whole time axis in one group -- the usual case -- the group offsets are all
    # zero.  Here the split is forced (dd_set_tuning) to 1, 2 and 3 tiles over 7 tiles and a ragged 8th: first tile
    # and first unit of a group != 0, a ragged last group, both buffers, one and two beams, device and host paths.
    full = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]]
    tb = 5120 if nbits == 2 else 3072
    cfg = full.reduced(nsamps=7 * tb + 555, ndm=21, nchans=40, nbeams=nbeams)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    dev = packed.cuda()
    out = torch.full((nbeams, cfg.ndm, cfg.nsamps), -1, dtype=torch.int32, device="cuda")
    h_out = torch.full((nbeams, cfg.ndm, cfg.nsamps), -1, dtype=torch.int32).pin_memory()
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=4) as p:
        p.set_tuning(dd.DD_TUNE_PAIR_TILES, tiles_per_group)
        p.set_dm_list(cfg.dm_list())
        if nbeams > 1:
            p.set_batch(nbeams, dev.stride(0), out.stride(0) * 4)
        p.execute(cfg.nsamps, dev, stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        info = p.launch_info()
        ngroups = -(-8 // tiles_per_group)
        assert info["variant"] == 4 and info["time_block"] == tb and info["last_launches"] == 1 + 2 * ngroups * nbeams
        assert p.workspace_bytes > 0
        p.execute_host(cfg.nsamps, packed.contiguous().pin_memory(), stride, h_out, -32)
    for b in range(nbeams):
        ref = oracle.dedisperse(packed[b].numpy(), cfg.nbits, cfg.nsamps, tab)
        got = out[b].cpu().numpy().view(np.uint32)
        bad = np.nonzero(got != ref)
        assert bad[0].size == 0, f"beam {b}: {bad[0].size} mismatches, first at d={bad[0][0]} t={bad[1][0]}"
        assert np.array_equal(h_out[b].numpy().view(np.uint32), ref)


def test_variant4_workspace_limit_splits_the_time_axis_and_is_worked_out_once():
    # dd_set_workspace_limit: a limit below the rows of the whole time axis makes the launcher split it (more launches,
    # same result); a limit below one tile's rows is an out-of-memory error, not a crash; the split is kept between calls
    cfg = W.CONFIGS[4].reduced(nsamps=6 * 3072 + 100, ndm=20, nchans=64)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    dev = packed.cuda()
    ref = oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab)
    out = torch.full((cfg.ndm, cfg.nsamps), -1, dtype=torch.int32, device="cuda")
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=4) as p:
        p.set_dm_list(cfg.dm_list())
        p.execute(cfg.nsamps, dev, stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert p.launch_info()["last_launches"] == 3 and np.array_equal(out.cpu().numpy().view(np.uint32), ref)
        whole = p.workspace_bytes
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=4) as p:
        p.set_dm_list(cfg.dm_list())
        p.set_workspace_limit(whole // 3)
        for _ in range(2):
            out.fill_(-1)
            p.execute(cfg.nsamps, dev, stride, out, -32, torch.cuda.current_stream())
            torch.cuda.synchronize()
            assert p.launch_info()["last_launches"] > 3 and np.array_equal(out.cpu().numpy().view(np.uint32), ref)
        assert p.workspace_bytes < whole
        p.set_workspace_limit(1024)
        with pytest.raises(dd.DDError):
            p.execute(cfg.nsamps, dev, stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        p.set_workspace_limit(0)     # and the plan still works afterwards
        p.execute(cfg.nsamps, dev, stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy().view(np.uint32), ref)


@pytest.mark.parametrize("nbeams", [1, 2])
@pytest.mark.parametrize("tiles_per_group", [1, 3])
@pytest.mark.parametrize("nbits,G", [(2, 4), (4, 4), (4, 2), (8, 4), (8, 2)])
def test_variant6_group_rows_and_time_axis_split(nbits, G, tiles_per_group, nbeams):
    # group rows in device memory (the default for 4- and 8-bit plans): rows of four (or two) channels per tuple of
    # delay differences, made group of time tiles by group on two internal streams.  The split is forced to 1 and 3
    # tiles over 7 tiles and a ragged 8th (first tile / first unit of a group != 0, ragged last group, both buffers),
    # one and two beams, device and host paths, every element against the oracle.
    full = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]]
    tb = 5120 if nbits == 2 else 3072
    cfg = full.reduced(nsamps=7 * tb + 555, ndm=21, nchans=42, nbeams=nbeams)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    dev = packed.cuda()
    out = torch.full((nbeams, cfg.ndm, cfg.nsamps), -1, dtype=torch.int32, device="cuda")
    h_out = torch.full((nbeams, cfg.ndm, cfg.nsamps), -1, dtype=torch.int32).pin_memory()
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=6) as p:
        p.set_tuning(dd.DD_TUNE_GROUP_SIZE, G).set_tuning(dd.DD_TUNE_PAIR_TILES, tiles_per_group)
        p.set_dm_list(cfg.dm_list())
        if nbeams > 1:
            p.set_batch(nbeams, dev.stride(0), out.stride(0) * 4)
        p.execute(cfg.nsamps, dev, stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        info = p.launch_info()
        ngroups = -(-8 // tiles_per_group)
        assert info["variant"] == 6 and info["time_block"] == tb and info["last_launches"] == 1 + 2 * ngroups * nbeams
        p.execute_host(cfg.nsamps, packed.contiguous().pin_memory(), stride, h_out, -32)
    for b in range(nbeams):
        ref = oracle.dedisperse(packed[b].numpy(), cfg.nbits, cfg.nsamps, tab)
        got = out[b].cpu().numpy().view(np.uint32)
        bad = np.nonzero(got != ref)
        assert bad[0].size == 0, f"beam {b}: {bad[0].size} mismatches, first at d={bad[0][0]} t={bad[1][0]}"
        assert np.array_equal(h_out[b].numpy().view(np.uint32), ref)


@pytest.mark.parametrize("nbits,G", [(2, 4), (4, 4), (4, 2), (8, 4), (8, 2)])
def test_variant6_group_rows_shapes_masks_and_dm_lists(nbits, G):
    # several tiles with a ragged tail and all output types; channel counts that leave partial and padded groups; the
    # high-DM end of the list (largest spreads, most tuples); a kill mask; an unsorted DM list
    full = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]]
    tb = 5120 if nbits == 2 else 3072

    def run(cfg, dms=None, kinds=("u32",), mask=None):
        dms = cfg.dm_list() if dms is None else np.asarray(dms, dtype=np.float64)
        tab = _oracle_table(cfg, dms)
        packed, stride = W.gen_packed(cfg, int(tab.max()))
        dev = packed.cuda()
        with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=6) as p:
            p.set_tuning(dd.DD_TUNE_GROUP_SIZE, G)
            p.set_killmask(mask)
            p.set_dm_list(dms)
            for kind in kinds:
                out = torch.full((1, len(dms), cfg.nsamps), -1, dtype=_TORCH_OUT[kind], device="cuda")
                p.execute(cfg.nsamps, dev, stride, out, {"f32": 32, "u32": -32, "u16": 16}[kind], torch.cuda.current_stream())
                torch.cuda.synchronize()
                assert p.launch_info()["variant"] == 6
                ref = oracle.cast_out(oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab, mask=mask), kind)
                got = out[0].cpu().numpy().view(_NP_VIEW[kind])
                bad = np.nonzero(got != ref)
                assert bad[0].size == 0, f"{cfg.name} G={G} {kind}: {bad[0].size} mismatches, first d={bad[0][0]} t={bad[1][0]}"

    run(full.reduced(nsamps=2 * tb + 333, ndm=37, nchans=200, nbeams=1), kinds=("f32", "u32") + (("u16",) if nbits < 8 else ()))
    for nchans in (1, 3, 17, 65):
        run(full.reduced(nsamps=1283, ndm=3, nchans=nchans, nbeams=1))
    cfg = full.reduced(nsamps=3000, ndm=40, nbeams=1)
    run(cfg, dms=np.asarray(full.dm_list())[-40:], kinds=("f32",))
    run(cfg, mask=(np.arange(cfg.nchans) % 4 != 1).astype(np.int32))
    small = full.reduced(nsamps=1000, ndm=24, nchans=96, nbeams=1)
    run(small, dms=np.asarray(small.dm_list())[np.random.default_rng(4).permutation(small.ndm)])


_GS_SHAPES = {2: [(2, 16), (4, 4)], 4: [(2, 8), (4, 4)], 8: [(2, 4), (2, 2), (4, 2), (4, 1)]}


def _gs_run(cfg, G, cc, dms=None, kind="u32", mask=None, host=False):
    dms = cfg.dm_list() if dms is None else np.asarray(dms, dtype=np.float64)
    tab = _oracle_table(cfg, dms)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    dev = packed.cuda()
    out = torch.full((cfg.nbeams, len(dms), cfg.nsamps), -1, dtype=_TORCH_OUT[kind], device="cuda")
    h_out = torch.full((cfg.nbeams, len(dms), cfg.nsamps), -1, dtype=_TORCH_OUT[kind]).pin_memory() if host else None
    code = {"f32": 32, "u32": -32, "u16": 16}[kind]
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=5) as p:
        p.set_tuning(dd.DD_TUNE_GROUP_SIZE, G).set_tuning(dd.DD_TUNE_GROUPS_PER_STAGE, cc)
        p.set_killmask(mask)
        p.set_dm_list(dms)
        if cfg.nbeams > 1:
            p.set_batch(cfg.nbeams, dev.stride(0), out.stride(0) * out.element_size())
        p.execute(cfg.nsamps, dev, stride, out, code, torch.cuda.current_stream())
        torch.cuda.synchronize()
        info = p.launch_info()
        assert info["variant"] == 5 and info["last_launches"] == 2 and info["chans_per_stage"] == cc
        if host:
            p.execute_host(cfg.nsamps, packed.contiguous().pin_memory(), stride, h_out, code)
    got = out.cpu().numpy().view(_NP_VIEW[kind])
    for b in range(cfg.nbeams):
        ref = oracle.cast_out(oracle.dedisperse(packed[b].numpy(), cfg.nbits, cfg.nsamps, tab, mask=mask), kind)
        bad = np.nonzero(got[b] != ref)
        assert bad[0].size == 0, (f"{cfg.name} G={G} cc={cc} {kind} beam {b}: {bad[0].size} mismatches, first at "
                                  f"d={bad[0][0]} t={bad[1][0]} got={got[b][bad[0][0], bad[1][0]]} ref={ref[bad[0][0], bad[1][0]]}")
        if host:
            assert np.array_equal(h_out[b].numpy().view(_NP_VIEW[kind]), ref)


@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_variant5_group_sums_in_shared_memory(nbits):
    # group sums made inside the CTA: every compiled shape (pairs and groups of four, two stage sizes each) on several
    # tiles with a ragged tail; channel counts that leave partial and padded groups; all output types; two beams
    # through device and host paths; the high-DM end of the list (largest spreads, most patterns); a kill mask; an
    # unsorted DM list (many patterns per block)
    full = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]]
    tb = 3072 if nbits == 2 else 2048
    for G, cc in _GS_SHAPES[nbits]:
        _gs_run(full.reduced(nsamps=2 * tb + 333, ndm=37, nchans=200, nbeams=1), G, cc)
        for nchans in (1, 3, 17, 65):
            _gs_run(full.reduced(nsamps=1283, ndm=3, nchans=nchans, nbeams=1), G, cc)
    G, cc = _GS_SHAPES[nbits][-2 if nbits == 8 else -1]
    _gs_run(full.reduced(nsamps=3000, ndm=40, nbeams=2), G, cc, kind="f32", host=True)
    cfg = full.reduced(nsamps=3000, ndm=40, nbeams=1)
    _gs_run(cfg, G, cc, dms=np.asarray(full.dm_list())[-40:], kind="f32")
    _gs_run(cfg, G, cc, mask=(np.arange(cfg.nchans) % 4 != 1).astype(np.int32), kind="u16" if nbits < 8 else "f32")
    G, cc = _GS_SHAPES[nbits][0]
    small = full.reduced(nsamps=1000, ndm=24, nchans=96, nbeams=1)
    _gs_run(small, G, cc, dms=np.asarray(small.dm_list())[np.random.default_rng(4).permutation(small.ndm)])


def test_variant2_channel_counts_around_group_and_flush_boundaries():
    # nchans not a multiple of 5 (group), of 40 (stage), beyond 85 (8-bit flush) and 17*5*k boundaries
    for nchans in (1, 4, 5, 6, 39, 41, 84, 85, 86, 171, 1023):
        _full_compare(W.CONFIGS[2].reduced(nsamps=1283, ndm=3, nchans=nchans), out_kinds=["u32"], variant=2)


@pytest.mark.parametrize("variant", [1, 2, 3, 4])
def test_cfg2_high_dm_end(variant):
    # the last DMs of config 2 (largest delays and spreads), nsamps not a multiple of 4
    cfg = W.CONFIGS[2].reduced(nsamps=1501, ndm=40)
    _full_compare(cfg, dms=W.CONFIGS[2].dm_list()[-40:], out_kinds=["f32", "u16"], variant=variant)


@pytest.mark.parametrize("variant", [1, 3])
def test_cfg3_reduced_8bit_4096_channels(variant):
    _full_compare(W.CONFIGS[3].reduced(nsamps=1300, ndm=33), variant=variant)


@pytest.mark.parametrize("variant", [1, 3])
def test_cfg3_high_dm_end_large_spread(variant):
    cfg = W.CONFIGS[3].reduced(nsamps=700, ndm=32)
    _full_compare(cfg, dms=W.CONFIGS[3].dm_list()[-32:], variant=variant)


@pytest.mark.parametrize("variant", [1, 3, 4])
def test_cfg4_reduced_4bit_u16(variant):
    _full_compare(W.CONFIGS[4].reduced(nsamps=2000, ndm=65), out_kinds=["u16", "u32", "f32"], variant=variant)


@pytest.mark.parametrize("variant", [1, 3])
def test_cfg5_reduced_batch_of_beams(variant):
    _full_compare(W.CONFIGS[5].reduced(nsamps=1000, ndm=40, nbeams=3), variant=variant)


@pytest.mark.parametrize("nbits", [4, 8])
def test_variant3_bitplane_4_and_8_bit_tiles_and_channel_padding(nbits):
    # bit-plane kernel, 4 planes per sub-row: 3072-sample tiles (2 tiles + ragged tail), 16-DM blocks (ragged),
    # all output types; channel counts around the stage size (16 / 8 channels, padded with zero channels) and the
    # ring depth; nsamps chosen so that 8-bit rows end in a half unit (16 bytes)
    base = W.CONFIGS[{4: 4, 8: 5}[nbits]]
    _full_compare(base.reduced(nsamps=2 * 3072 + 333, ndm=37, nchans=96), out_kinds=["f32", "u32", "u16"], variant=3)
    for nchans in (1, 7, 8, 9, 15, 16, 17, 33, 63, 65, 257):
        _full_compare(base.reduced(nsamps=1283, ndm=3, nchans=nchans), out_kinds=["u32"], variant=3)
    _full_compare(base.reduced(nsamps=3072 + 8, ndm=2, nchans=5), out_kinds=["u32"], variant=3)


@pytest.mark.parametrize("tpc", [0, 1, 2, 3, 8])
@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_variant3_short_plans_walk_several_time_tiles_per_cta(nbits, tpc):
    # plans with few channels (the short instantiation of the bit-plane kernel: step 2 of the sub-band method, small
    # transforms) let a CTA walk several consecutive time tiles with the ring of stages running on across them:
    # 7 tiles and a ragged 8th, 1 / 2 / 3 / 8 tiles per CTA (ragged last CTA), the library's own choice, two beams,
    # all output types, every element against the oracle
    full = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]]
    tb = 5120 if nbits == 2 else 3072
    cfg = full.reduced(nsamps=7 * tb + 555, ndm=21, nchans=40, nbeams=2)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    dev = packed.cuda()
    for kind in (["u32", "f32"] + (["u16"] if nbits < 8 else [])):
        out = torch.full((2, cfg.ndm, cfg.nsamps), -1, dtype=_TORCH_OUT[kind], device="cuda")
        with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=3) as p:
            p.set_tuning(dd.DD_TUNE_TILES_PER_CTA, tpc)
            p.set_dm_list(cfg.dm_list())
            p.set_batch(2, dev.stride(0), out.stride(0) * out.element_size())
            p.execute(cfg.nsamps, dev, stride, out, {"f32": 32, "u32": -32, "u16": 16}[kind], torch.cuda.current_stream())
            torch.cuda.synchronize()
            assert p.launch_info()["variant"] == 3
        got = out.cpu().numpy().view(_NP_VIEW[kind])
        for b in range(2):
            ref = oracle.cast_out(oracle.dedisperse(packed[b].numpy(), cfg.nbits, cfg.nsamps, tab), kind)
            bad = np.nonzero(got[b] != ref)
            assert bad[0].size == 0, f"{kind} beam {b}: {bad[0].size} mismatches, first at d={bad[0][0]} t={bad[1][0]}"


@pytest.mark.parametrize("nbits", [4, 8])
def test_variant3_bitplane_4_and_8_bit_extreme_values(nbits):
    # every sample at its maximum with the largest channel count the planes hold: 4369 * 15 = 65535 (all 16
    # planes set); 4112 * 255 = 1048560 (the top of the 20-plane range); and all zero
    nchans = {4: 4369, 8: 4112}[nbits]
    base = W.CONFIGS[{4: 4, 8: 3}[nbits]]
    cfg = W.Config(name="extreme", index=base.index, nchans=nchans, f_top=base.f_top, df=-100.0 / nchans, dt=base.dt,
                   nbits=nbits, nsamps=700, ndm=5, dm_max=20.0, out="u32", dist="uniform", seed=7)
    tab = _oracle_table(cfg)
    nbytes = ((cfg.nsamps + int(tab.max())) * nbits + 7) // 8
    stride = (nbytes + 15) // 16 * 16
    for fill, want in ((0xFF, nchans * ((1 << nbits) - 1)), (0x00, 0)):
        packed = torch.full((1, cfg.nchans, stride), fill, dtype=torch.uint8)
        got = _gpu_transform(cfg, packed.cuda(), stride, cfg.dm_list(), "u32", cfg.nsamps, 3)
        ref = oracle.dedisperse(packed[0].numpy(), nbits, cfg.nsamps, tab)
        assert np.array_equal(got[0], ref) and int(ref.max()) == want and int(ref.min()) == want


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_odd_shapes(nbits, variant):
    # channel count not a multiple of the stage size, one DM, tiny nsamps, more channels than a flush interval
    base = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]]
    for nchans, ndm, nsamps in ((1, 1, 1), (37, 5, 13), (300, 33, 641), (1024, 2, 5)):
        _full_compare(base.reduced(nsamps=nsamps, ndm=ndm, nchans=nchans), out_kinds=["u32"], variant=variant)


def test_unsorted_dm_list():
    cfg = W.CONFIGS[2].reduced(nsamps=900, ndm=48, nchans=256)
    rng = np.random.default_rng(11)
    dms = rng.permutation(W.CONFIGS[2].dm_list()[:200])[:48]
    _full_compare(cfg, dms=dms, out_kinds=["f32"])


def test_many_channels_need_32bit_accumulators():
    # 2-bit, 24000 channels: 24000*3 > 65535 -> the 32-bit accumulator instantiation
    cfg = W.Config(name="wide32", index=2, nchans=24000, f_top=1500.0, df=-0.01, dt=64e-6, nbits=2, nsamps=333,
                   ndm=3, dm_max=2.0, out="u32", dist="uniform", seed=99)
    _full_compare(cfg)
    cfg4 = W.Config(name="wide32-4", index=4, nchans=5000, f_top=1500.0, df=-0.05, dt=64e-6, nbits=4, nsamps=200,
                    ndm=2, dm_max=1.0, out="u32", dist="uniform", seed=98)
    _full_compare(cfg4)


@pytest.mark.parametrize("variant", [0, 1, 2, 3])   # variant 4 with a kill mask: test_variant4_pair_rows
def test_killmask_every_variant(variant):
    # PAPER.md:113 kill mask against the oracle's arithmetic form (sum += data * mask[c]); masks that kill
    # runs, single channels, the first and the last channel, so that the live list is ragged against the stage size
    cfg = W.CONFIGS[2].reduced(nsamps=5120 + 700, ndm=21, nchans=200)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    dev = packed.cuda()
    rng = np.random.default_rng(113)
    masks = [(rng.random(cfg.nchans) < 0.7).astype(np.int32), np.zeros(cfg.nchans, np.int32), None]
    masks[0][[0, cfg.nchans - 1]] = 0
    masks[0][50:90] = 0
    for mask in masks:
        out = torch.full((cfg.ndm, cfg.nsamps), -1, dtype=torch.int32, device="cuda")
        with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=variant) as p:
            p.set_dm_list(cfg.dm_list())
            p.set_killmask(mask)                   # after the DM list: tiles rebuilt at once
            p.execute(cfg.nsamps, dev[0], stride, out, -32, torch.cuda.current_stream())
            torch.cuda.synchronize()
        ref = oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab, mask=mask)
        assert np.array_equal(out.cpu().numpy().view(np.uint32), ref)


@pytest.mark.parametrize("nbits", [4, 8])
def test_killmask_4_and_8_bit_batch_and_host_path(nbits):
    cfg = W.CONFIGS[{4: 4, 8: 5}[nbits]].reduced(nsamps=3072 + 100, ndm=18, nchans=77, nbeams=2)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    dev = packed.cuda()
    mask = (np.arange(cfg.nchans) % 3 != 1).astype(np.int32)
    out = torch.full((2, cfg.ndm, cfg.nsamps), -1, dtype=torch.float32, device="cuda")
    h_out = torch.zeros((2, cfg.ndm, cfg.nsamps), dtype=torch.float32).pin_memory()
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_killmask(mask)                       # before the DM list
        p.set_dm_list(cfg.dm_list())
        p.set_batch(2, dev.stride(0), out.stride(0) * 4)
        p.execute(cfg.nsamps, dev, stride, out, 32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        p.execute_host(cfg.nsamps, packed.contiguous().pin_memory(), stride, h_out, 32)
    for b in range(2):
        ref = oracle.dedisperse(packed[b].numpy(), cfg.nbits, cfg.nsamps, tab, mask=mask).astype(np.float32)
        assert np.array_equal(out[b].cpu().numpy(), ref)
        assert np.array_equal(h_out[b].numpy(), ref)


@pytest.mark.parametrize("case", [
    # (config, nchans, ndm, nsamps, sb_nchans, dm_group, nbeams, masked)
    (2, 256, 50, 5120 + 333, 32, 16, 1, False),     # 2-bit, ragged last group of trials, two time tiles
    (2, 256, 70, 1500, 64, 32, 2, True),            # two beams, kill mask, ragged last group
    (2, 96, 33, 700, 8, 16, 1, False),              # sub-bands smaller than a stage (padded groups)
    (2, 1024, 48, 2000, 1, 16, 1, False),           # 1-channel sub-bands: the direct transform through 2 steps
    (4, 64, 40, 3072 + 50, 16, 16, 1, True),        # 4-bit: 16 * 15 = 240 <= 255
    (5, 48, 35, 900, 1, 32, 1, False),              # 8-bit input: only 1-channel sub-bands fit 8-bit intermediates
])
@pytest.mark.parametrize("gpc", [0, 3])   # sub-bands summed per CTA in step 1: the library's choice / forced to 3
def test_subband_method_matches_the_two_step_oracle(case, gpc):
    idx, nchans, ndm, nsamps, sb, grp, nbeams, masked = case
    cfg = W.CONFIGS[idx].reduced(nsamps=nsamps, ndm=ndm, nchans=nchans, nbeams=nbeams)
    dms = cfg.dm_list()
    nominal, d1, d2 = oracle.subband_tables(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms, sb, grp)
    extent = oracle.subband_required_samples(nsamps, d1, d2, sb) - nsamps
    packed, stride = W.gen_packed(cfg, max(extent, int(_oracle_table(cfg).max())))
    dev = packed.cuda()
    mask = (np.arange(nchans) % 7 != 3).astype(np.int32) if masked else None
    out = torch.full((nbeams, ndm, nsamps), -1, dtype=torch.int32, device="cuda")
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_tuning(dd.DD_TUNE_SUBBAND_GPC, gpc)
        p.set_dm_list(dms)
        p.set_killmask(mask)
        p.set_subband(sb, grp)
        assert p.subband_extent == extent
        g_nom, g_d1, g_d2 = p.subband_tables()
        assert np.array_equal(g_nom, nominal) and np.array_equal(g_d1, d1) and np.array_equal(g_d2, d2)
        if nbeams > 1:
            p.set_batch(nbeams, dev.stride(0), out.stride(0) * 4)
        p.execute(nsamps, dev, stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert p.launch_info()["last_launches"] == 3    # pre-pass, step 1 (writes bit planes), step 2
        got = out.cpu().numpy().view(np.uint32)
        for b in range(nbeams):
            ref = oracle.subband_dedisperse(packed[b].numpy(), cfg.nbits, nsamps, cfg.nchans, cfg.dt, cfg.f_top, cfg.df,
                                            dms, sb, grp, mask=mask)
            assert np.array_equal(got[b], ref), f"beam {b}"
        if gpc == 0:      # the same through the host-buffer path (one time slab on the staged copy)
            h_out = torch.full((nbeams, ndm, nsamps), -1, dtype=torch.int32).pin_memory()
            p.execute_host(nsamps, packed.contiguous().pin_memory(), stride, h_out, -32)
            assert np.array_equal(h_out.numpy().view(np.uint32), got)
        if sb == 1:       # and that IS the direct transform
            assert np.array_equal(got[0], oracle.dedisperse(packed[0].numpy(), cfg.nbits, nsamps, _oracle_table(cfg)))
        # back to the direct transform on the same plan
        p.set_subband(0, 0)
        p.execute(nsamps, dev, stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        ref = oracle.dedisperse(packed[0].numpy(), cfg.nbits, nsamps, _oracle_table(cfg), mask=mask)
        assert np.array_equal(out[0].cpu().numpy().view(np.uint32), ref)


@pytest.mark.parametrize("widths", [(2, 4), (2, 8), (4, 8)])
def test_time_scrunch_and_dedispersion_of_the_scrunched_series(widths):
    # pairs of samples added; then the scrunched rows go through a plan made with 2*dt
    nin, nout = widths
    base = W.CONFIGS[2 if nin == 2 else 4]
    nchans, ndm, ns2 = 64, 20, 2000 + 37                       # scrunched output samples per DM trial
    cfg2x = W.Config(name="scrunched", index=base.index, nchans=nchans, f_top=base.f_top, df=base.df, dt=2 * base.dt,
                     nbits=nout, nsamps=ns2, ndm=ndm, dm_max=400.0, out="u32", dist="uniform", seed=71)
    tab2 = _oracle_table(cfg2x)                                # delays in units of 2*dt
    n2 = ns2 + int(tab2.max())                                 # scrunched samples per row
    src = base.reduced(nsamps=2 * n2, ndm=1, nchans=nchans)    # 2*n2 raw samples per row, no extra delay
    packed, stride = W.gen_packed(src, 64)
    out_stride = ((n2 * nout + 7) // 8 + 15) // 16 * 16
    dev_in = packed[0].cuda()
    dev_s = torch.zeros((nchans, out_stride), dtype=torch.uint8, device="cuda")
    dd.dd_time_scrunch(nchans, n2, dev_in, stride, nin, dev_s, out_stride, nout, torch.cuda.current_stream())
    torch.cuda.synchronize()
    want = oracle.time_scrunch(packed[0].numpy(), nin, n2)      # unpacked int64 sums
    got = oracle.unpack(dev_s.cpu().numpy(), nout, n2).astype(np.int64)
    assert np.array_equal(got, want) and int(want.max()) == 2 * ((1 << nin) - 1)
    # the scrunched rows through the transform at half the time resolution
    out = torch.full((ndm, ns2), -1, dtype=torch.int32, device="cuda")
    with dd.Plan(nchans, cfg2x.dt, cfg2x.f_top, cfg2x.df, nout) as p:
        p.set_dm_list(cfg2x.dm_list())
        p.execute(ns2, dev_s, out_stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
    ref = oracle.dedisperse_unpacked(want.astype(np.uint8), ns2, tab2)
    assert np.array_equal(out.cpu().numpy().view(np.uint32), ref)


@pytest.mark.parametrize("case", [
    # (config, nchans, nsamps, max_factor, DM list)
    (2, 96, 4000 + 37, 64, [0.0, 30.0, 90.0, 150.0, 155.0, 290.0, 400.0, 640.0, 990.0, 1000.0]),   # 2-bit: factors 1..8
    (2, 1024, 2048, 4, [0.0, 60.0, 70.0, 200.0, 999.0]),                                          # capped at 4
    (4, 64, 3100, 64, [0.0, 100.0, 300.0, 700.0, 1500.0, 1999.0, 2000.0]),                        # 4-bit: up to 16
    (5, 32, 900, 64, [0.0, 500.0, 1000.0]),                                                       # 8-bit: one level
])
def test_scrunched_transform_matches_the_oracle_level_by_level(case):
    # pairs of samples added beyond 2x, 4x, ... the diagonal DM; every level bit-exact
    idx, nchans, nsamps, max_factor, dms = case
    base = W.CONFIGS[idx]
    cfg = base.reduced(nsamps=nsamps, ndm=len(dms), nchans=nchans)
    dms = np.asarray(dms, dtype=np.float64)
    with dd.ScrunchSet(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, dms, max_factor) as s:
        lv = s.levels
        need_bytes = s.required_bytes(nsamps)
        nsamp_in = need_bytes * 8 // cfg.nbits
        packed, stride = W.gen_packed(cfg, nsamp_in - nsamps)
        assert stride >= need_bytes
        ref = oracle.scrunched_dedisperse(packed[0].numpy(), cfg.nbits, nsamps, cfg.nchans, cfg.dt, cfg.f_top, cfg.df,
                                          dms, max_factor, nsamp_in)
        assert [l["factor"] for l in lv] == [F for F, _, _ in ref]
        if idx == 2 and nchans == 96:
            assert [l["factor"] for l in lv] == [1, 2, 4, 8]
        dev = packed[0].cuda()
        outs = [torch.full((l["ndm"], nsamps // l["factor"]), -1, dtype=torch.int32, device="cuda") for l in lv]
        for rep in range(2):                               # the second call reuses the set's buffers
            s.execute(nsamps, dev, stride, outs, -32, torch.cuda.current_stream())
            torch.cuda.synchronize()
            for l, o, (F, first, want) in zip(lv, outs, ref):
                assert l["first_dm"] == first
                assert np.array_equal(o.cpu().numpy().view(np.uint32), want.astype(np.uint32)), f"factor {F}"
        f_outs = [torch.zeros((l["ndm"], nsamps // l["factor"]), dtype=torch.float32, device="cuda") for l in lv]
        s.execute(nsamps, dev, stride, f_outs, 32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        for o, (F, first, want) in zip(f_outs, ref):
            assert np.array_equal(o.cpu().numpy(), want.astype(np.float32))
        with pytest.raises(dd.DDError):                    # rows shorter than the set needs
            s.execute(nsamps, dev, 16, outs, -32, None)
        mask = (np.arange(cfg.nchans) % 6 != 4).astype(np.int32)         # kill mask at every level
        s.set_killmask(mask)
        s.execute(nsamps, dev, stride, outs, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        ref_m = oracle.scrunched_dedisperse(packed[0].numpy(), cfg.nbits, nsamps, cfg.nchans, cfg.dt, cfg.f_top, cfg.df,
                                            dms, max_factor, nsamp_in, mask=mask)
        for o, (F, first, want) in zip(outs, ref_m):
            assert np.array_equal(o.cpu().numpy().view(np.uint32), want.astype(np.uint32)), f"masked, factor {F}"


@pytest.mark.parametrize("case", [(8, 160, 24), (8, 160, 48), (8, 136, 100), (8, 40, 30), (8, 40, 200), (4, 528, 6), (4, 48, 5)])
def test_input_max_promise_skips_planes_but_not_results(case):
    # dd_set_input_max: samples <= vmax -> the instantiation that leaves out the planes that cannot be set
    # (long instantiations: 8-bit with >= 128 channels, 4-bit with >= 512; short ones below that)
    nbits, nchans, vmax = case
    base = W.CONFIGS[5 if nbits == 8 else 4]
    cfg = base.reduced(nsamps=3072 + 100, ndm=19, nchans=nchans)
    tab = _oracle_table(cfg)
    nsamp_in = (cfg.nsamps + int(tab.max()) + 127) // 128 * 128
    rng = np.random.default_rng(1000 * nbits + vmax)
    vals = rng.integers(0, vmax + 1, size=(nchans, nsamp_in), dtype=np.int64)
    vals[:, ::97] = vmax                                                      # the largest value does occur
    packed = W.pack_rows(torch.from_numpy(vals.astype(np.uint8)), nbits).contiguous()
    stride = packed.shape[1]
    ref = oracle.dedisperse(packed.numpy(), nbits, cfg.nsamps, tab)
    out = torch.full((cfg.ndm, cfg.nsamps), -1, dtype=torch.int32, device="cuda")
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, nbits) as p:
        p.set_dm_list(cfg.dm_list()).set_input_max(vmax)
        p.execute(cfg.nsamps, packed.cuda(), stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy().view(np.uint32), ref.astype(np.uint32))
        p.set_input_max(0)                                                    # promise withdrawn: same result
        out.fill_(-1)
        p.execute(cfg.nsamps, packed.cuda(), stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy().view(np.uint32), ref.astype(np.uint32))
        with pytest.raises(dd.DDError):
            p.set_input_max(1 << nbits)


@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_u16_rows_that_are_not_16_byte_aligned(nbits):
    # regression: uint16 rows of nsamps % 8 == 4 samples start on 8-byte, not 16-byte boundaries; the coalescing
    # epilogue of the bit-plane kernel stores 16 bytes at a time and must leave such rows to the plain path
    idx = {2: 2, 4: 4, 8: 5}[nbits]
    tb = 5120 if nbits == 2 else 3072
    cfg = W.CONFIGS[idx].reduced(nsamps=tb + 4, ndm=5, nchans=32)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    ref = oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab)
    out = torch.zeros((cfg.ndm, cfg.nsamps), dtype=torch.int16, device="cuda")
    h_out = torch.zeros((cfg.ndm, cfg.nsamps), dtype=torch.int16).pin_memory()
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(cfg.dm_list())
        p.execute(cfg.nsamps, packed[0].cuda(), stride, out, 16, torch.cuda.current_stream())
        torch.cuda.synchronize()
        p.execute_host(cfg.nsamps, packed[0].contiguous().pin_memory(), stride, h_out, 16)
    assert np.array_equal(out.cpu().numpy().view(np.uint16), ref.astype(np.uint16))
    assert np.array_equal(h_out.numpy().view(np.uint16), ref.astype(np.uint16))


@pytest.mark.parametrize("variant", [0, 1, 2, 4])
@pytest.mark.parametrize("pad", [16, 1])   # rows padded by 16 elements (16-byte aligned rows) / by one element
def test_output_row_stride(variant, pad):
    # PAPER.md:388 "arbitrary strides through the ... output arrays": rows out_dm_stride bytes apart, padding untouched
    cfg = W.CONFIGS[2].reduced(nsamps=5120 + 40, ndm=19, nchans=40, nbeams=2)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    dev = packed.cuda()
    pitch = cfg.nsamps + pad
    for tdtype, code, es in ((torch.float32, 32, 4), (torch.int16, 16, 2)):
        out = torch.full((2, cfg.ndm, pitch), -7, dtype=tdtype, device="cuda")
        h_out = torch.full((2, cfg.ndm, pitch), -7, dtype=tdtype).pin_memory()
        with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=variant) as p:
            p.set_dm_list(cfg.dm_list()).set_output_stride(pitch * es)
            p.set_batch(2, dev.stride(0), out.stride(0) * es)
            p.execute(cfg.nsamps, dev, stride, out, code, torch.cuda.current_stream())
            torch.cuda.synchronize()
            p.execute_host(cfg.nsamps, packed.contiguous().pin_memory(), stride, h_out, code)
        for b in range(2):
            ref = oracle.dedisperse(packed[b].numpy(), cfg.nbits, cfg.nsamps, tab)
            for o in (out[b].cpu(), h_out[b]):
                assert np.array_equal(o[:, :cfg.nsamps].numpy().astype(np.int64), ref)
                assert bool((o[:, cfg.nsamps:] == -7).all())          # the padding between rows was not written


def test_output_row_stride_subband_and_all_killed():
    cfg = W.CONFIGS[2].reduced(nsamps=1500, ndm=40, nchans=64)
    dms = cfg.dm_list()
    nominal, d1, d2 = oracle.subband_tables(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms, 16, 16)
    extent = oracle.subband_required_samples(cfg.nsamps, d1, d2, 16) - cfg.nsamps
    packed, stride = W.gen_packed(cfg, max(extent, int(_oracle_table(cfg).max())))
    pitch = cfg.nsamps + 20
    out = torch.full((cfg.ndm, pitch), -7, dtype=torch.int32, device="cuda")
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(dms).set_output_stride(pitch * 4)
        p.set_subband(16, 16)
        p.execute(cfg.nsamps, packed[0].cuda(), stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        ref = oracle.subband_dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms, 16, 16)
        assert np.array_equal(out[:, :cfg.nsamps].cpu().numpy().view(np.uint32), ref.astype(np.uint32))
        assert bool((out[:, cfg.nsamps:] == -7).all())
        p.set_subband(0, 0)
        p.set_killmask(np.zeros(cfg.nchans, dtype=np.int32))      # every channel killed: zeros, padding untouched
        out.fill_(-7)
        p.execute(cfg.nsamps, packed[0].cuda(), stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert bool((out[:, :cfg.nsamps] == 0).all()) and bool((out[:, cfg.nsamps:] == -7).all())


def test_execute_host_matches_oracle():
    cfg = W.CONFIGS[4].reduced(nsamps=2 * 640 + 100, ndm=40, nchans=256)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    ref = oracle.cast_out(oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab), "u16")
    out = torch.zeros((cfg.ndm, cfg.nsamps), dtype=torch.int16).pin_memory()
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(cfg.dm_list())
        p.execute_host(cfg.nsamps, packed[0].contiguous().pin_memory(), stride, out, 16)
    assert np.array_equal(out.numpy().view(np.uint16), ref)


def test_execute_host_bitplane_variant_two_slabs():
    # 2-bit through the host-buffer path: 140000 output samples = two time slabs (133120 + ragged rest)
    cfg = W.CONFIGS[2].reduced(nsamps=140000, ndm=9, nchans=64)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    ref = oracle.cast_out(oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab), "f32")
    out = torch.zeros((cfg.ndm, cfg.nsamps), dtype=torch.float32).pin_memory()
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=3) as p:
        p.set_dm_list(cfg.dm_list())
        p.set_tuning(dd.DD_TUNE_HOST_SLAB, 1 << 17)
        p.execute_host(cfg.nsamps, packed[0].contiguous().pin_memory(), stride, out, 32)
        assert p.launch_info()["last_launches"] == 4
        assert np.array_equal(out.numpy(), ref)
        # the default slabs (2^15 samples rounded up to 7 tiles of 5120: four slabs); the bytes of every row the first
        # slab reads are copied in first, the rest of the rows behind them
        out.zero_()
        p.set_tuning(dd.DD_TUNE_HOST_SLAB, 0)
        p.execute_host(cfg.nsamps, packed[0].contiguous().pin_memory(), stride, out, 32)
        assert p.launch_info()["last_launches"] == 8
    assert np.array_equal(out.numpy(), ref)


@pytest.mark.parametrize("nbits,dense", [(2, True), (4, False), (8, True)])
def test_execute_host_many_slabs_fresh_staging(nbits, dense):
    # first call of a fresh plan (its staging buffer has never held the input): slabs of one and of three tiles, so that
    # the first slab's kernels run while most of the rows are still on their way; two beams whose rows lie back to back
    # (the head of all rows is one strided copy) or apart (one copy of everything); the library's default kernel
    full = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]]
    cfg = full.reduced(nsamps=60000, ndm=21, nchans=160, nbeams=2)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    gap = 0 if dense else 4 * stride
    h_in = torch.zeros((cfg.nbeams, cfg.nchans * stride + gap), dtype=torch.uint8).pin_memory()
    h_in[:, :cfg.nchans * stride] = packed.reshape(cfg.nbeams, -1)
    for slab in (1, 15000):
        h_out = torch.full((cfg.nbeams, cfg.ndm, cfg.nsamps), -1, dtype=torch.int32).pin_memory()
        with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
            p.set_dm_list(cfg.dm_list())
            p.set_batch(cfg.nbeams, h_in.stride(0), h_out.stride(0) * 4)
            p.set_tuning(dd.DD_TUNE_HOST_SLAB, slab)
            p.execute_host(cfg.nsamps, h_in, stride, h_out, -32)
        for b in range(cfg.nbeams):
            ref = oracle.dedisperse(packed[b].numpy(), cfg.nbits, cfg.nsamps, tab)
            assert np.array_equal(h_out[b].numpy().view(np.uint32), ref), (nbits, dense, slab, b)


def test_execute_host_bitplane_8bit_two_slabs():
    # 8-bit through the host-buffer path: two time slabs, rows ending in a half unit
    cfg = W.CONFIGS[5].reduced(nsamps=140008, ndm=5, nchans=24)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    ref = oracle.cast_out(oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab), "f32")
    out = torch.zeros((cfg.ndm, cfg.nsamps), dtype=torch.float32).pin_memory()
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=3) as p:
        p.set_dm_list(cfg.dm_list())
        p.set_tuning(dd.DD_TUNE_HOST_SLAB, 1 << 17)
        p.execute_host(cfg.nsamps, packed[0].contiguous().pin_memory(), stride, out, 32)
        assert p.launch_info()["last_launches"] == 4
    assert np.array_equal(out.numpy(), ref)


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("nbits", [2, 8])
def test_dm_slab_and_time_slab_shards_through_the_kernel(nbits, world):
    # the two exchange-free splits besides beams, driven through dd_execute on one GPU,
    # one "rank" after the other: DM slabs (own plan with the slab's DM sub-list, input replicated) and time slabs
    # (input pointer advanced to the slab's first byte, nsamps = slab length, a halo of max_delay samples read by both
    # neighbours); the shards are reassembled and compared with the oracle on every element.  Ragged last slabs.
    from paper_1201_5380_b200 import multi
    full = W.CONFIGS[{2: 2, 8: 5}[nbits]]
    cfg = full.reduced(nsamps=5 * 1024 + 700, ndm=53, nchans=72, nbeams=1)
    dms = cfg.dm_list()
    tab = _oracle_table(cfg)
    max_delay = int(tab.max())
    packed, stride = W.gen_packed(cfg, max_delay)
    ref = oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab)
    # rows must be readable out to in_stride from the advanced pointer: one spare row behind the last channel
    dev = torch.cat([packed[0], torch.zeros((1, stride), dtype=torch.uint8)]).cuda()
    st = torch.cuda.current_stream()
    # DM slabs
    got = torch.full((cfg.ndm, cfg.nsamps), -1, dtype=torch.int32, device="cuda")
    covered = 0
    for rank in range(world):
        lo, hi = multi.shard_dm_slabs(cfg.ndm, world, rank)
        assert lo % 16 == 0 and lo == covered
        covered = hi
        if hi == lo:
            continue
        with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
            p.set_dm_list(dms[lo:hi])
            p.execute(cfg.nsamps, dev, stride, got[lo:hi], -32, st)
            torch.cuda.synchronize()
    assert covered == cfg.ndm and np.array_equal(got.cpu().numpy().view(np.uint32), ref)
    # time slabs, each written in place through the output row stride
    got.fill_(-1)
    covered = 0
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(dms)
        p.set_output_stride(cfg.nsamps * 4)
        for rank in range(world):
            t_lo, t_hi, in_lo, in_hi = multi.shard_time_slabs(cfg.nsamps, world, rank, max_delay)
            assert t_lo == covered and in_lo == t_lo and in_hi == t_hi + max_delay and (t_lo * cfg.nbits) % 128 == 0
            covered = t_hi
            if t_hi == t_lo:
                continue
            p.execute(t_hi - t_lo, dev.data_ptr() + t_lo * cfg.nbits // 8, stride, got.data_ptr() + 4 * t_lo, -32, st)
            torch.cuda.synchronize()
    assert covered == cfg.nsamps and np.array_equal(got.cpu().numpy().view(np.uint32), ref)


def test_device_generation_equals_host_generation():
    cfg = W.CONFIGS[2].reduced(nsamps=5000, ndm=8, nchans=64)
    a, s1 = W.gen_packed(cfg, 300)
    b, s2 = W.gen_packed(cfg, 300, device="cuda")
    assert s1 == s2 and torch.equal(a, b.cpu())
    cfg = W.CONFIGS[3].reduced(nsamps=3000, ndm=8, nchans=32)
    a, _ = W.gen_packed(cfg, 100)
    b, _ = W.gen_packed(cfg, 100, device="cuda")
    assert torch.equal(a, b.cpu())


# ------------------------------------------------------- full BASELINE.json sizes, sampled by the oracle
def _sample_points(cfg, tile, n, seed):
    rng = np.random.default_rng(seed)
    d = rng.integers(0, cfg.ndm, n)
    t = rng.integers(0, cfg.nsamps, n)
    # structured points: first/last DM, tile edges, last samples
    edge_t = [0, 1, tile - 1, tile, tile + 1, cfg.nsamps - tile - 1, cfg.nsamps - 2, cfg.nsamps - 1]
    edge_d = [0, 1, 31, 32, 33, cfg.ndm - 33, cfg.ndm - 2, cfg.ndm - 1]
    dd_, tt = np.meshgrid(np.clip(edge_d, 0, cfg.ndm - 1), np.clip(edge_t, 0, cfg.nsamps - 1))
    return np.concatenate([d, dd_.ravel()]), np.concatenate([t, tt.ravel()])


def _compare_block(cfg, out_b, packed_host, tab, rows, t0, length, what):
    """Every output of the trials `rows` over the samples [t0, t0 + length) against the C oracle run on the packed rows
    from sample t0 on (t0 * nbits is a whole number of bytes: tiles are multiples of 1024 samples)."""
    rows = np.asarray(rows, dtype=np.int64)
    byte0 = t0 * cfg.nbits // 8
    byte1 = min(packed_host.shape[1], -(-(t0 + length + int(tab[rows].max())) * cfg.nbits // 8) + 16)
    sub = packed_host if byte0 == 0 and byte1 == packed_host.shape[1] else np.ascontiguousarray(packed_host[:, byte0:byte1])
    ref = oracle.cast_out(oracle.dedisperse(sub, cfg.nbits, length, tab[rows]), cfg.out)
    got = out_b[torch.as_tensor(rows, device="cuda"), t0:t0 + length].cpu().numpy().view(_NP_VIEW[cfg.out])
    bad = np.nonzero(got != ref)
    assert bad[0].size == 0, (f"{cfg.name} {what}: {bad[0].size}/{ref.size} outputs differ; first d={rows[bad[0][0]]} "
                              f"t={t0 + bad[1][0]} got={got[bad[0][0], bad[1][0]]} ref={ref[bad[0][0], bad[1][0]]}")
    return ref.size


def _full_size_sampled(cfg, npoints, whole_rows=0, everything=False, blocks_and_tiles=False):
    """The transform at the full BASELINE.json size in the configuration bench.py times, against the oracle:
    sampled outputs (random + tile / block edges) evaluated one by one; `whole_rows` whole DM rows; `everything`:
    every output element (cfg2: ~16 s of oracle on 16 host threads); `blocks_and_tiles`: every output of three whole
    16-trial DM blocks (first, middle, last -- the last has the largest delay spread) over the whole time axis, and
    every trial over the first and the last (ragged or not) time tile, for the first and the last beam."""
    tab = _oracle_table(cfg)
    pulses = W.make_pulses(cfg, lambda idx: tab[idx])
    max_delay = int(tab.max())
    packed_dev, stride = W.gen_packed(cfg, max_delay, pulses, device="cuda", chan_chunk=16)
    got_dev_out = None
    nbeams, ndm, nsamps = cfg.nbeams, cfg.ndm, cfg.nsamps
    out = torch.full((nbeams, ndm, nsamps), -1, dtype=_TORCH_OUT[cfg.out], device="cuda")
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(cfg.dm_list())
        tile = p.launch_info()["time_block"]
        if nbeams > 1:
            p.set_batch(nbeams, packed_dev.stride(0), out.stride(0) * out.element_size())
        p.execute(nsamps, packed_dev, stride, out, cfg.out_nbits, torch.cuda.current_stream())
        torch.cuda.synchronize()
    for b in sorted({0, nbeams - 1}):
        d_idx, t_idx = _sample_points(cfg, tile, npoints, seed=cfg.seed + b)
        ref = oracle.dedisperse_points(
            lambda c, t: W.values_at(cfg, b, c, t, pulses).numpy(), tab, d_idx, t_idx)
        got = out[b][torch.as_tensor(d_idx, device="cuda"), torch.as_tensor(t_idx, device="cuda")].cpu().numpy()
        got = got.view(_NP_VIEW[cfg.out]).astype(np.int64)
        bad = np.nonzero(got != ref)[0]
        assert bad.size == 0, (f"{cfg.name} beam {b}: {bad.size}/{ref.size} sampled outputs differ; first "
                               f"d={d_idx[bad[0]]} t={t_idx[bad[0]]} got={got[bad[0]]} ref={ref[bad[0]]}")
    if whole_rows:
        rows = np.unique(np.concatenate([np.linspace(0, ndm - 1, whole_rows).astype(np.int64), [ndm - 1]]))
        packed_host = packed_dev[0].cpu().numpy()
        ref_rows = oracle.cast_out(oracle.dedisperse(packed_host, cfg.nbits, nsamps, tab[rows]), cfg.out)
        got_rows = out[0][torch.as_tensor(rows, device="cuda")].cpu().numpy().view(_NP_VIEW[cfg.out])
        assert np.array_equal(got_rows, ref_rows)
    compared = 0
    if everything or blocks_and_tiles:
        for b in sorted({0, nbeams - 1}):
            packed_host = packed_dev[b].cpu().numpy()
            if everything:
                for r0 in range(0, ndm, 96):
                    compared += _compare_block(cfg, out[b], packed_host, tab, np.arange(r0, min(r0 + 96, ndm)), 0, nsamps,
                                               f"beam {b} trials {r0}..")
            else:
                nblk = -(-ndm // 16)
                for blk in sorted({0, nblk // 2, nblk - 1}):
                    compared += _compare_block(cfg, out[b], packed_host, tab, np.arange(blk * 16, min(blk * 16 + 16, ndm)), 0,
                                               nsamps, f"beam {b} DM block {blk}")
                ntiles = -(-nsamps // tile)
                for tl in sorted({0, ntiles - 1}):
                    t0 = tl * tile
                    for r0 in range(0, ndm, 512):
                        compared += _compare_block(cfg, out[b], packed_host, tab, np.arange(r0, min(r0 + 512, ndm)), t0,
                                                   min(tile, nsamps - t0), f"beam {b} time tile {tl}")
            del packed_host
        print(f"{cfg.name}: {compared} outputs compared element by element")
    # every element was written (the buffer was pre-filled with -1 / NaN-like patterns)
    if cfg.out == "f32":
        assert bool((out >= 0).all())
    del out, packed_dev
    torch.cuda.empty_cache()


def test_cfg2_full_size_bench_configuration_every_element():
    _full_size_sampled(W.CONFIGS[2], npoints=4000, everything=True)


def test_cfg3_full_size_blocks_tiles_and_samples():
    _full_size_sampled(W.CONFIGS[3], npoints=1500, blocks_and_tiles=True)


def test_cfg4_full_size_blocks_tiles_and_samples():
    _full_size_sampled(W.CONFIGS[4], npoints=3000, blocks_and_tiles=True)


def test_cfg5_full_size_batch_blocks_tiles_and_samples():
    _full_size_sampled(W.CONFIGS[5], npoints=2000, blocks_and_tiles=True)


def test_cfg2_full_size_subband_32_32_sampled():
    # the sub-band method at the size bench.py --subband 32,32 times: sampled outputs against the direct sum with
    # the summed delays delta1 + delta2 (the identity pinned by P13), evaluated one output at a time
    cfg, sb, grp = W.CONFIGS[2], 32, 32
    dms = cfg.dm_list()
    nominal, d1, d2 = oracle.subband_tables(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms, sb, grp)
    summed = d1[np.arange(cfg.ndm) // grp] + np.repeat(d2, sb, axis=1)            # [ndm][nchans]
    extent = oracle.subband_required_samples(cfg.nsamps, d1, d2, sb) - cfg.nsamps
    assert int(summed.max()) <= extent
    packed_dev, stride = W.gen_packed(cfg, max(extent, int(_oracle_table(cfg).max())), None, device="cuda", chan_chunk=16)
    out = torch.full((cfg.ndm, cfg.nsamps), -1, dtype=torch.float32, device="cuda")
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(dms)
        p.set_subband(sb, grp)
        assert p.subband_extent == extent
        p.execute(cfg.nsamps, packed_dev[0], stride, out, 32, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert p.launch_info()["last_launches"] == 3
    d_idx, t_idx = _sample_points(cfg, 3072, 3000, seed=321)
    ref = oracle.dedisperse_points(lambda c, t: W.values_at(cfg, 0, c, t, None).numpy(), summed, d_idx, t_idx)
    got = out[torch.as_tensor(d_idx, device="cuda"), torch.as_tensor(t_idx, device="cuda")].cpu().numpy().astype(np.int64)
    bad = np.nonzero(got != ref)[0]
    assert bad.size == 0, f"{bad.size}/{ref.size} differ; first d={d_idx[bad[0]]} t={t_idx[bad[0]]} got={got[bad[0]]} ref={ref[bad[0]]}"
    assert bool((out >= 0).all())                                                  # every element was written
    del out, packed_dev
    torch.cuda.empty_cache()


def test_cfg2_full_size_scrunched_sampled():
    # the transform with time-scrunching at the size bench.py --scrunch 16 times: sampled outputs of every level,
    # D_F[d][t] = sum_c sum_{i<F} A[c][F (t + delay_F[d][c]) + i], one output at a time
    cfg = W.CONFIGS[2]
    dms = np.asarray(cfg.dm_list())
    with dd.ScrunchSet(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, dms, 16) as s:
        lv = s.levels
        assert [l["factor"] for l in lv] == [1, 2, 4, 8, 16]
        need = s.required_bytes(cfg.nsamps)
        packed_dev, stride = W.gen_packed(cfg, need * 8 // cfg.nbits - cfg.nsamps, None, device="cuda", chan_chunk=16)
        outs = [torch.full((l["ndm"], cfg.nsamps // l["factor"]), -1, dtype=torch.float32, device="cuda") for l in lv]
        s.execute(cfg.nsamps, packed_dev[0], stride, outs, 32, torch.cuda.current_stream())
        torch.cuda.synchronize()
    rng = np.random.default_rng(99)
    for l, o in zip(lv, outs):
        F, ns = l["factor"], cfg.nsamps // l["factor"]
        tabF = oracle.delay_table(cfg.nchans, cfg.dt * F, cfg.f_top, cfg.df, dms[l["first_dm"]:l["first_dm"] + l["ndm"]])
        assert int(tabF.max()) == l["max_delay"]
        d_idx = np.concatenate([rng.integers(0, l["ndm"], 400), [0, l["ndm"] - 1, 0, l["ndm"] - 1]])
        t_idx = np.concatenate([rng.integers(0, ns, 400), [0, 0, ns - 1, ns - 1]])
        ref = np.zeros(d_idx.shape[0], dtype=np.int64)
        for i in range(F):
            ref += oracle.dedisperse_points(lambda c, t: W.values_at(cfg, 0, c, t, None).numpy(), tabF * F, d_idx, t_idx * F + i)
        got = o[torch.as_tensor(d_idx, device="cuda"), torch.as_tensor(t_idx, device="cuda")].cpu().numpy().astype(np.int64)
        bad = np.nonzero(got != ref)[0]
        assert bad.size == 0, f"factor {F}: {bad.size}/{ref.size} differ; first d={d_idx[bad[0]]} t={t_idx[bad[0]]}"
        assert bool((o >= 0).all())
    del outs, packed_dev
    torch.cuda.empty_cache()


def test_dd_execute_and_scrunch_set_are_cuda_graph_capturable():
    # dd_execute neither allocates nor synchronises after its first call, so a warmed-up call can be captured into
    # a CUDA graph and replayed on new input (launch-bound cases: small transforms, the 14 launches of a scrunch set)
    cfg = W.CONFIGS[2].reduced(nsamps=5120 + 77, ndm=21, nchans=64)
    tab = _oracle_table(cfg)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    cfg_b = W.CONFIGS[2].reduced(nsamps=5120 + 77, ndm=21, nchans=64, nbeams=2)
    other, _ = W.gen_packed(cfg_b, int(tab.max()), beams=[1])          # a second, different input of the same shape
    dev = packed[0].cuda()
    out = torch.zeros((cfg.ndm, cfg.nsamps), dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(cfg.dm_list())
        with torch.cuda.stream(side):
            p.execute(cfg.nsamps, dev, stride, out, 32, side)          # warm-up: tables uploaded, work buffer grown
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            p.execute(cfg.nsamps, dev, stride, out, 32, torch.cuda.current_stream())
        for src in (packed[0], other[0], packed[0]):
            dev.copy_(src.cuda())
            out.zero_()
            g.replay()
            torch.cuda.synchronize()
            ref = oracle.dedisperse(src.numpy(), cfg.nbits, cfg.nsamps, tab)
            assert np.array_equal(out.cpu().numpy(), ref.astype(np.float32))
    # the group-row launcher (8-bit input, >= 128 channels) forks onto internal streams and joins them: capturable too
    cfg8 = W.CONFIGS[5].reduced(nsamps=3072 + 200, ndm=20, nchans=160, nbeams=2)
    tab8 = _oracle_table(cfg8)
    pk8, st8 = W.gen_packed(cfg8, int(tab8.max()))
    dev8 = pk8.cuda()
    out8 = torch.zeros((2, cfg8.ndm, cfg8.nsamps), dtype=torch.float32, device="cuda")
    with dd.Plan(cfg8.nchans, cfg8.dt, cfg8.f_top, cfg8.df, cfg8.nbits) as p:
        p.set_dm_list(cfg8.dm_list())
        assert p.launch_info()["variant"] == 6
        p.set_batch(2, dev8.stride(0), out8.stride(0) * 4)
        with torch.cuda.stream(side):
            p.execute(cfg8.nsamps, dev8, st8, out8, 32, side)
        side.synchronize()
        g8 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g8, stream=side):
            p.execute(cfg8.nsamps, dev8, st8, out8, 32, torch.cuda.current_stream())
        out8.zero_()
        g8.replay()
        torch.cuda.synchronize()
        for b in range(2):
            ref8 = oracle.dedisperse(pk8[b].numpy(), cfg8.nbits, cfg8.nsamps, tab8)
            assert np.array_equal(out8[b].cpu().numpy(), ref8.astype(np.float32))
    dms = np.array([0.0, 100.0, 300.0, 900.0])
    with dd.ScrunchSet(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, dms, 8) as s:
        lv = s.levels
        need = s.required_bytes(cfg.nsamps)
        nsamp_in = need * 8 // cfg.nbits
        pk, st2 = W.gen_packed(cfg, nsamp_in - cfg.nsamps)
        dev2 = pk[0].cuda()
        outs = [torch.zeros((l["ndm"], cfg.nsamps // l["factor"]), dtype=torch.float32, device="cuda") for l in lv]
        with torch.cuda.stream(side):
            s.execute(cfg.nsamps, dev2, st2, outs, 32, side)
        side.synchronize()
        g2 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g2, stream=side):
            s.execute(cfg.nsamps, dev2, st2, outs, 32, torch.cuda.current_stream())
        for o in outs:
            o.zero_()
        g2.replay()
        torch.cuda.synchronize()
        ref = oracle.scrunched_dedisperse(pk[0].numpy(), cfg.nbits, cfg.nsamps, cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms, 8, nsamp_in)
        assert len(ref) == len(outs) >= 3
        for o, (F, first, want) in zip(outs, ref):
            assert np.array_equal(o.cpu().numpy(), want.astype(np.float32)), f"factor {F}"


@pytest.mark.parametrize("case", [
    # (config, nchans, ndm, nsamps, keep one channel in ..., expected variant)
    (5, 512, 40, 3500, 3, 6), (4, 1024, 64, 4000, 4, 6), (5, 300, 1200, 2000, 2, 6), (3, 4096, 32, 1500, 7, 3),
    (5, 64, 20, 1500, 1, 3),
])
def test_default_variant_for_4_and_8_bit_input_under_sparse_kill_masks(case):
    # plans of >= 128 channels take group rows (variant 6) by default when its cost model says they pay, also when a
    # sparse kill mask groups channels that are far apart; when the rows do not pay or fit (cfg3's largest DMs, one
    # channel in seven kept) or the plan is small, the library falls back to variant 3 -- the same result each way
    idx, nchans, ndm, nsamps, mod, want_variant = case
    cfg = W.CONFIGS[idx].reduced(nsamps=nsamps, ndm=ndm, nchans=nchans, nbeams=1)
    dms = W.CONFIGS[3].dm_list()[-32:] if idx == 3 else cfg.dm_list()
    tab = _oracle_table(cfg, dms)
    packed, stride = W.gen_packed(cfg, int(tab.max()))
    mask = (np.arange(nchans) % mod == 0).astype(np.int32)
    ref = oracle.dedisperse(packed[0].numpy(), cfg.nbits, nsamps, tab, mask=mask)
    out = torch.full((len(dms), nsamps), -1, dtype=torch.int32, device="cuda")
    with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits) as p:
        p.set_dm_list(dms)
        p.set_killmask(mask)
        assert p.launch_info()["variant"] == want_variant
        p.execute(nsamps, packed[0].cuda(), stride, out, -32, torch.cuda.current_stream())
        torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy().view(np.uint32), ref.astype(np.uint32))
