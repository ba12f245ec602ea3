"""GPU parity of the tree dedispersion algorithm and the piecewise linear tree method
(PAPER.md:181-222): dd_tree_execute through the C ABI against oracle.tree / oracle.piecewise_tree, element by element,
bit-exact.  The oracle follows eq. 10-15 / 18-23 step by step and is pinned by P16 / P17 (tests/test_oracle_pins.py).
All inputs are seeded and synthetic (dd_workloads); no expected value comes from the CUDA path.
"""
from dataclasses import replace

import numpy as np
import pytest
import torch

import dd_workloads as W
import oracle
import paper_1201_5380_b200 as dd

pytestmark = pytest.mark.gpu

_CODE = {"f32": 32, "u32": -32, "u16": 16}
_TORCH_OUT = {"f32": torch.float32, "u32": torch.int32, "u16": torch.int16}
_NP_VIEW = {"f32": np.float32, "u32": np.uint32, "u16": np.uint16}


def _band(nbits, nchans, nsamps):
    """A one-beam config on the survey band (cfg2's) with the value distribution of the config of that width."""
    base = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]]
    return base.reduced(nsamps=nsamps, ndm=2, nchans=nchans, nbeams=1)


def _run(tree, nsamps, packed_dev, stride, nrows, kind):
    out = torch.full((nrows, nsamps), -1, dtype=_TORCH_OUT[kind], device="cuda")
    tree.execute(nsamps, packed_dev, stride, out, _CODE[kind], torch.cuda.current_stream())
    torch.cuda.synchronize()
    return out.cpu().numpy().view(_NP_VIEW[kind])


def _assert_equal(got, ref, what):
    assert got.shape == ref.shape, what
    bad = np.nonzero(got != ref)
    assert bad[0].size == 0, (f"{what}: {bad[0].size} mismatches, first at row {bad[0][0]} t {bad[1][0]}: "
                              f"got {got[bad[0][0], bad[1][0]]} ref {ref[bad[0][0], bad[1][0]]}")


def _tree_case(nbits, n, nsamps, kinds=("u32",), tuning=()):
    cfg = _band(nbits, n, nsamps)
    packed, stride = W.gen_packed(cfg, n - 1, None)
    ref = oracle.tree(packed[0].numpy(), nbits, nsamps)
    dev = packed.cuda()
    with dd.Tree(n, n, nbits) as t:
        for key, value in tuning:
            t.set_tuning(key, value)
        assert t.required_samples(nsamps) == nsamps + n - 1
        for kind in kinds:
            got = _run(t, nsamps, dev, stride, n, kind)
            _assert_equal(got, oracle.cast_out(ref, kind), f"tree N={n} {nbits}-bit {kind} tuning {tuning}")
        info = t.info()
        assert info["last_launches"] == info["passes"] >= 1 and sum(info["steps"]) == n.bit_length() - 1
    return info


@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_tree_every_size_one_and_two_passes(nbits):
    # N = 2 .. 64: one pass; 128 .. 4096: two.  Four tiles of the first pass and a ragged tail; a row
    # length that allows 16-byte stores and one that does not; all output types
    for n in (2, 4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048, 4096):
        wide = n * ((1 << nbits) - 1) > 65535        # 8-bit samples, 512 channels and more: 32-bit lanes throughout
        kinds = ("u16", "u32", "f32") if n in (4, 64, 256) else (("u32", "f32") if n == 1024 else ("u32",))
        info = _tree_case(nbits, n, 4 * 448 + 77, kinds)
        assert info["passes"] == (1 if n <= (32 if wide else 64) else 2 if n <= (1024 if wide else 4096) else 3)
        if wide:                                     # sums that do not fit uint16 rows are refused at execute
            with dd.Tree(n, n, nbits) as t, pytest.raises(dd.DDError) as err:
                t.execute(64, torch.zeros(16, dtype=torch.uint8, device="cuda"), 1 << 20, torch.zeros(16, device="cuda"), 16)
            assert err.value.status == -6
    _tree_case(nbits, 64, 2048, ("u16", "f32"))
    for k6 in (1, 2, 3):
        _tree_case(nbits, 64, 2048, ("u32",), tuning=((6, k6),))
        _tree_case(nbits, 512, 3000, ("u32",), tuning=((6, k6),))


def test_tree_later_passes_over_several_tiles():
    # 256 channels: the second pass (two steps) stores 8128 columns per tile; 40000 samples are five of its tiles
    info = _tree_case(2, 256, 40000)
    assert info["passes"] == 2 and info["tile"][1] < 10000
    info = _tree_case(4, 1024, 7000)       # second pass (four steps, rows staged skewed): tiles of 1984 of 2048 columns
    assert info["steps"] == [6, 4] and info["tile"] == [384, 1984]
    info = _tree_case(4, 1024, 7000, tuning=((3, 8), (4, 8)))   # one CTA per SM: twice the columns
    assert info["steps"] == [6, 4] and info["tile"] == [896, 4032]
    info = _tree_case(2, 2048, 9000)       # 8-bit rows between the passes, five steps in the second: 960 of 1024 columns
    assert info["steps"] == [6, 5] and info["tile"] == [896, 960]
    info = _tree_case(4, 4096, 3000, tuning=((1, 3), (2, 3)))   # four passes: every row is stored early for the next one
    assert info["steps"] == [3, 3, 3, 3]


@pytest.mark.parametrize("first", [1, 2, 3, 4, 5, 6])
def test_tree_pass_shapes(first):
    # every radix of the pass kernel as first pass (packed input) and as later pass (16-bit rows), both thread loads
    # (2-bit samples: 8-bit lanes in the first pass unless told otherwise; 4-bit: only while 15 * 2^first < 256)
    for later in (1, 2, 3):
        for items, nbits, lanes in ((4, 4, 0), (8, 2, 0), (4, 2, 16), (8, 4, 16)):
            # (key 6: bit 0 = the first two steps in shared memory instead of in registers while staging, bit 1 = one step
            # per trip through shared memory instead of two)
            info = _tree_case(nbits, 64, 1500, tuning=((1, first), (2, later), (3, items), (4, items), (5, lanes), (6, (first + later) % 4)))
            assert info["steps"][0] == first and all(s <= later for s in info["steps"][1:])
    for later in (4, 5, 6):
        if first + later <= 8:
            _tree_case(2, 256, 1100, tuning=((1, first), (2, later)))


def _piecewise_case(nbits, nchans, sb, ndm, dm_hi, nsamps, kind="u32", tuning=()):
    cfg = _band(nbits, nchans, nsamps)
    dms = np.linspace(0.0, dm_hi, ndm)
    with dd.Tree(nchans, sb, nbits) as t:
        for key, value in tuning:
            t.set_tuning(key, value)
        t.set_dm_list(cfg.dt, cfg.f_top, cfg.df, dms)
        dprime, dt2 = t.tables()
        need = t.required_samples(nsamps)
        assert need == nsamps + int(dt2.max()) + sb - 1 and int(dprime.max()) < sb
        packed, stride = W.gen_packed(cfg, need - nsamps, None)
        got = _run(t, nsamps, packed.cuda(), stride, ndm, kind)
        info = t.info()
        assert info["last_launches"] == info["passes"] + 1
    ref = oracle.piecewise_tree(packed[0].numpy(), nbits, nsamps, nchans, cfg.dt, cfg.f_top, cfg.df, dms, sb)
    _assert_equal(got, oracle.cast_out(ref, kind), f"piecewise tree {nchans}/{sb} {nbits}-bit {kind}")
    return dprime, dt2


@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_piecewise_linear_tree_small_bands(nbits):
    # sub-bands of 8 .. 64 channels, trials up to just below the diagonal DM of the last sub-band, several tiles of both stages
    dprime, _ = _piecewise_case(nbits, 256, 32, 23, 45.0, 2 * 960 + 501, "u32")
    assert dprime.max() >= 20                      # the trials do reach far into the trees
    _piecewise_case(nbits, 256, 8, 9, 50.0, 3000, "f32")
    _piecewise_case(nbits, 128, 64, 17, 68.0, 2111, "u16" if nbits < 8 else "u32")
    _piecewise_case(nbits, 64, 64, 5, 70.0, 1000)   # one sub-band: stage 2 only picks rows
    if nbits == 8:                                  # sub-bands of 512 eight-bit channels: 32-bit lanes in both stages
        _piecewise_case(8, 1024, 512, 9, 40.0, 1500, "f32")
    # stage-1 rows in 16-bit lanes where the default is 8-bit lanes (2-bit samples), and two passes of stage 1
    _piecewise_case(nbits, 256, 32, 23, 45.0, 2000, "u16" if nbits < 8 else "u32", tuning=((5, 16),))
    _piecewise_case(nbits, 128, 64, 17, 68.0, 1500, "f32", tuning=((1, 3), (2, 3)))


def test_piecewise_linear_tree_survey_band_and_the_diagonal():
    # cfg2's band (1024 channels, 2-bit) in sub-bands of 32: the trials of its DM list below the diagonal DM
    cfg = W.CONFIGS[2]
    step = cfg.dm_max / (cfg.ndm - 1)
    dprime, dt2 = _piecewise_case(2, 1024, 32, 40, 39 * step, 5000, "f32")
    assert dprime.max() < 32 and dt2.max() > 500
    with dd.Tree(1024, 32, 2) as t:                 # one trial beyond the diagonal: an error, the tree unchanged
        t.set_dm_list(cfg.dt, cfg.f_top, cfg.df, [0.0, 10.0])
        with pytest.raises(dd.DDError) as err:
            t.set_dm_list(cfg.dt, cfg.f_top, cfg.df, [0.0, 10.0, 200.0])
        assert err.value.status == -6
        assert t.tables()[0].shape == (2, 32)


def test_tree_full_size_survey_band_windows():
    # cfg2's shape: 1024 channels, 2-bit, 2^19 samples, float32 rows.  The transform is invariant under time shifts, so the
    # oracle is run on windows of the input: the start, the joints of the tiles of both passes, the end
    n, nbits, nsamps, win = 1024, 2, 1 << 19, 1536
    cfg = _band(nbits, n, nsamps)
    packed, stride = W.gen_packed(cfg, n - 1, None)
    dev = packed.cuda()
    with dd.Tree(n, n, nbits) as t:
        got = _run(t, nsamps, dev, stride, n, "f32")
        info = t.info()
        torch.cuda.synchronize()
    assert info["steps"] == [6, 4]
    starts = [0, 896 - 64, 1984 - 128, 100 * 1984 - 700, 273 * 896 - 512, nsamps - win]
    host = packed[0].numpy()
    for a in starts:
        assert a % 4 == 0
        rows = host[:, a // 4:(a + win + n - 1 + 3) // 4 + 1]
        ref = oracle.tree(np.ascontiguousarray(rows), nbits, win)
        _assert_equal(got[:, a:a + win], oracle.cast_out(ref, "f32"), f"window at {a}")
    # every row sums every channel once: the mean level of a row is the mean level of the band
    assert abs(float(got.mean()) - float(got[0].mean())) < 1.0


@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_frequency_padded_tree(nbits):
    # the real channels at the rows of eq. 25 of a stretched band of N_pad rows, blank rows between them,
    # one tree over all of it.  Bands that stretch by a few per cent and by 1.56 (the survey band's ratio), one to three passes
    for nchans, f_top, df, nsamps, kind in ((24, 1500.0, -8.0, 1111, "u32"), (100, 1581.8, -0.390625, 2 * 960 + 77, "u16"),
                                            (100, 1581.8, -4.0, 3000, "f32"), (1024, 1581.8, -0.390625, 2500, "f32")):
        cfg = W.CONFIGS[{2: 2, 4: 4, 8: 5}[nbits]].reduced(nsamps=nsamps, ndm=2, nchans=nchans, nbeams=1)
        with dd.Tree.padded(nchans, f_top, df, nbits) as t:
            npad = t.nchans
            assert t.required_samples(nsamps) == nsamps + npad - 1 and npad >= nchans
            packed, stride = W.gen_packed(cfg, npad - 1, None)
            got = _run(t, nsamps, packed.cuda(), stride, npad, kind)
            assert t.info()["last_launches"] == t.info()["passes"]
        ref = oracle.padded_tree(packed[0].numpy(), nbits, nsamps, f_top, df)
        _assert_equal(got, oracle.cast_out(ref, kind), f"padded tree {nchans} -> {npad} rows, {nbits}-bit {kind}")


@pytest.mark.parametrize("world", [2, 3])
def test_tree_time_slab_shards_reassemble(world):
    # PAPER.md:456 ("time-division multiplexing"): the tree is invariant under time shifts, so ranks take time
    # slabs with a halo of the samples the trails reach into (N - 1; max Dt'' + N' - 1 for the piecewise method), no
    # exchange.  One "rank" after the other on one GPU: input pointer advanced to the slab's first byte, nsamps = the slab's
    # length; the slabs side by side are the whole transform (ragged last slab).
    from paper_1201_5380_b200 import multi
    st = torch.cuda.current_stream()
    n, nbits, nsamps = 256, 2, 5 * 1024 + 700
    cfg = _band(nbits, n, nsamps)
    for piecewise in (False, True):
        with (dd.Tree(n, 32, nbits) if piecewise else dd.Tree(n, n, nbits)) as t:
            dms = np.linspace(0.0, 45.0, 19)
            if piecewise:
                t.set_dm_list(cfg.dt, cfg.f_top, cfg.df, dms)
            halo = t.required_samples(nsamps) - nsamps
            packed, stride = W.gen_packed(cfg, halo, None)
            ref = (oracle.piecewise_tree(packed[0].numpy(), nbits, nsamps, n, cfg.dt, cfg.f_top, cfg.df, dms, 32) if piecewise
                   else oracle.tree(packed[0].numpy(), nbits, nsamps))
            dev = torch.cat([packed[0], torch.zeros((1, stride), dtype=torch.uint8)]).cuda()   # (rows readable out to in_stride)
            parts, covered = [], 0
            for rank in range(world):
                t_lo, t_hi, in_lo, in_hi = multi.shard_time_slabs(nsamps, world, rank, halo)
                assert t_lo == covered and in_lo == t_lo and in_hi == t_hi + halo and (t_lo * nbits) % 128 == 0
                covered = t_hi
                if t_hi == t_lo:
                    continue
                out = torch.full((ref.shape[0], t_hi - t_lo), -1, dtype=torch.int32, device="cuda")
                t.execute(t_hi - t_lo, dev.data_ptr() + t_lo * nbits // 8, stride, out, _CODE["u32"], st)
                torch.cuda.synchronize()
                parts.append(out.cpu().numpy().view(np.uint32))
            assert covered == nsamps
            _assert_equal(np.concatenate(parts, axis=1), oracle.cast_out(ref, "u32"), f"time slabs, piecewise={piecewise}, world {world}")


def test_tree_execute_is_cuda_graph_capturable():
    # after its first call for a size dd_tree_execute only enqueues kernels (no allocation, no synchronisation): a warmed-up
    # call is captured into a CUDA graph and replayed on new input -- the tree (two passes) and the piecewise method
    n, nbits, nsamps = 256, 2, 3000
    cfg = _band(nbits, n, nsamps)
    side = torch.cuda.Stream()
    dms = np.linspace(0.0, 45.0, 11)
    for piecewise in (False, True):
        with (dd.Tree(n, 32, nbits) if piecewise else dd.Tree(n, n, nbits)) as t:
            if piecewise:
                t.set_dm_list(cfg.dt, cfg.f_top, cfg.df, dms)
            halo = t.required_samples(nsamps) - nsamps
            inputs = [W.gen_packed(replace(cfg, seed=cfg.seed + k), halo, None) for k in range(2)]
            stride = inputs[0][1]
            dev = inputs[0][0][0].cuda()
            out = torch.zeros((len(dms) if piecewise else n, nsamps), dtype=torch.float32, device="cuda")
            with torch.cuda.stream(side):
                t.execute(nsamps, dev, stride, out, _CODE["f32"], side)      # warm-up: rows between the passes, tables
            side.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                t.execute(nsamps, dev, stride, out, _CODE["f32"], torch.cuda.current_stream())
            for k in (0, 1, 0):
                dev.copy_(inputs[k][0][0].cuda())
                out.zero_()
                g.replay()
                torch.cuda.synchronize()
                host = inputs[k][0][0].numpy()
                ref = (oracle.piecewise_tree(host, nbits, nsamps, n, cfg.dt, cfg.f_top, cfg.df, dms, 32) if piecewise
                       else oracle.tree(host, nbits, nsamps))
                _assert_equal(out.cpu().numpy(), oracle.cast_out(ref, "f32"), f"graph replay {k}, piecewise={piecewise}")


def test_trees_of_several_beams_in_one_call():
    # the rows of three beams back to back (768 rows, trees of 256: not a power of two in all): one call, one tree per beam
    nbits, n, nbeams, nsamps = 2, 256, 3, 3000
    cfg = W.CONFIGS[2].reduced(nsamps=nsamps, ndm=2, nchans=n, nbeams=nbeams)
    packed, stride = W.gen_packed(cfg, n - 1, None)
    with dd.Tree(nbeams * n, n, nbits) as t:
        got = _run(t, nsamps, packed.cuda(), stride, nbeams * n, "u32")
    for b in range(nbeams):
        ref = oracle.tree(packed[b].numpy(), nbits, nsamps)
        _assert_equal(got[b * n:(b + 1) * n], oracle.cast_out(ref, "u32"), f"beam {b}")
