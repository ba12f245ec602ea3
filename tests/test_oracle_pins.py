"""Pins for the CPU oracle (oracle/) -- what the paper and the mathematics fix, NOT the oracle re-typed.

Pin numbering follows DESIGN.md section 3 (P1..P15).  None of these tests touches the CUDA path.

  P1  hand-evaluated eq. 1 delays (tests/golden/delays_eq1_hand.txt)
  P2  closed-form properties + exact rational arithmetic (fractions.Fraction)
  P3  table checksums computed independently for the survey
  P4  DM = 0 row is the plain channel sum (numpy.sum)                            eq. 5 with DM = 0
  P5  impulse response, brute force over (channel, time), all nbits              eq. 3
  P6  linearity                                                                   eq. 3 is a sum
  P7  time-shift covariance                                                       eq. 3
  P8  an injected dispersed pulse peaks at its own DM trial and time             PAPER.md:37 (Fig. 1)
  P9  C loop == numpy gather == pure-Python triple loop on tiny inputs           eq. 3
  P10 output statistics of uniform 2-bit noise                                   eq. 3 + CLT
  P11 packing convention: bytes 0xE4 / 0x21                                      reading R9
  P12 kill mask: equals the unmasked sum over zeroed rows; complements add up
  P13 sub-band method: reduces to the direct transform for 1-channel sub-bands; equals a direct transform with
      the summed delays; error of the summed delays within the analytic bound; impulse response
  P14 time-scrunching: hand example, conservation of the total, equals a reshape-sum
  P15 transform with time-scrunching: the diagonal DM in exact rational arithmetic (unit gradient at the end of the
      band); factor ranges by their definition; every level equals the pinned C loop at full resolution with the
      delays F * delay_F, summed over F consecutive outputs; max_factor 1 is the plain transform
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

import dd_workloads as W
import oracle


def _table(cfg):
    return oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.dm_list())


def _read_rows(path):
    rows = []
    with open(path) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows


# ----------------------------------------------------------------------------- P1
def test_p1_hand_delays(golden_dir):
    cfg = W.CONFIGS[1]
    for dm, c, x_hand, delay in _read_rows(os.path.join(golden_dir, "delays_eq1_hand.txt")):
        dm, c, x_hand, delay = float(dm), int(c), float(x_hand), int(delay)
        tab = oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, [dm])
        assert tab[0, c] == delay, (dm, c)
        assert abs(tab[0, c] - x_hand) <= 0.5 + 0.05
        assert round(x_hand) == delay


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("idx", [1, 2, 3, 4])
def test_p2_closed_form_properties(idx):
    cfg = W.CONFIGS[idx]
    tab = _table(cfg)
    assert tab.shape == (cfg.ndm, cfg.nchans)
    assert (tab[:, 0] == 0).all(), "delay is relative to the start of the band (PAPER.md:60)"
    assert (tab[0, :] == 0).all(), "DM = 0 has no delay (eq. 5)"
    assert (np.diff(tab, axis=1) >= 0).all(), "lower frequency arrives later (eq. 1)"
    assert (np.diff(tab, axis=0) >= 0).all(), "delay grows with DM (eq. 1)"
    assert tab.min() >= 0


def _exact_delay(cfg, dm: float, c: int) -> int:
    """floor(x + 1/2) with x evaluated in exact rational arithmetic on the double inputs."""
    K = Fraction(4148808, 1000)
    f_top, df, dt = Fraction(cfg.f_top), Fraction(cfg.df), Fraction(cfg.dt)
    f = f_top + c * df
    x = K * Fraction(dm) * (1 / (f * f) - 1 / (f_top * f_top)) / dt
    return math.floor(x + Fraction(1, 2))


def test_p2_exact_rational_full_cfg1():
    cfg = W.CONFIGS[1]
    tab = _table(cfg)
    dms = cfg.dm_list()
    for d in range(cfg.ndm):
        for c in range(cfg.nchans):
            assert tab[d, c] == _exact_delay(cfg, float(dms[d]), c), (d, c)


@pytest.mark.parametrize("idx", [2, 3, 4])
def test_p2_exact_rational_sampled(idx):
    cfg = W.CONFIGS[idx]
    tab = _table(cfg)
    dms = cfg.dm_list()
    rng = np.random.default_rng(idx)
    ds = np.concatenate([rng.integers(0, cfg.ndm, 1500), [0, 1, cfg.ndm - 1, cfg.ndm - 1]])
    cs = np.concatenate([rng.integers(0, cfg.nchans, 1500), [cfg.nchans - 1, 1, cfg.nchans - 1, 0]])
    for d, c in zip(ds, cs):
        assert tab[d, c] == _exact_delay(cfg, float(dms[d]), int(c)), (d, c)


def test_p2_k_dm_is_the_papers_constant():
    """The common 1/2.41e-4 approximation must NOT be what the oracle uses (reading R3)."""
    cfg = W.CONFIGS[2]
    tab = oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, [1000.0])
    f_lo = cfg.f_top + (cfg.nchans - 1) * cfg.df
    x_paper = 4.148808e3 * 1000.0 * (f_lo ** -2 - cfg.f_top ** -2) / cfg.dt
    x_approx = (1.0 / 2.41e-4) * 1000.0 * (f_lo ** -2 - cfg.f_top ** -2) / cfg.dt
    assert abs(x_paper - x_approx) > 2.0
    assert abs(tab[0, -1] - x_paper) <= 0.5


# ----------------------------------------------------------------------------- P3
def test_p3_table_checksums(golden_dir):
    for idx, mx, sm, mid in _read_rows(os.path.join(golden_dir, "table_checksums.txt")):
        cfg = W.CONFIGS[int(idx)]
        tab = _table(cfg)
        assert int(tab.max()) == int(mx)
        assert int(tab.sum()) == int(sm)
        if int(mid) >= 0:
            assert int(tab[cfg.ndm // 2, cfg.nchans // 2]) == int(mid)


def test_p3_two_evaluation_orders_agree():
    """north_star's expression (C oracle) and the paper's LUT order eq. 4 then eq. 5 (numpy) give one table (R2)."""
    for idx in (1, 2, 3, 4):
        cfg = W.CONFIGS[idx]
        assert np.array_equal(_table(cfg), oracle.delay_table_np(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.dm_list()))


# ----------------------------------------------------------------------- helpers
def _random_case(nbits, nchans, nsamps, ndm, maxdelay, seed):
    rng = np.random.default_rng(seed)
    delays = rng.integers(0, maxdelay + 1, size=(ndm, nchans)).astype(np.int64)
    delays[0, :] = 0
    per = 8 // nbits
    a_len = -(-(nsamps + maxdelay) // (16 * per)) * (16 * per)
    a = rng.integers(0, 1 << nbits, size=(nchans, a_len)).astype(np.uint8)
    packed = W.pack_rows(torch.from_numpy(a), nbits).numpy()
    return a, packed, delays


# ----------------------------------------------------------------------------- P4
@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_p4_dm0_is_channel_sum(nbits):
    a, packed, delays = _random_case(nbits, 37, 1000, 3, 50, seed=nbits)
    out = oracle.dedisperse(packed, nbits, 1000, delays)
    assert np.array_equal(out[0], a[:, :1000].astype(np.int64).sum(axis=0))


def test_p4_dm0_cfg1_real_table():
    cfg = W.CONFIGS[1]
    tab = _table(cfg)
    packed, _ = W.gen_packed(cfg, int(tab.max()))
    out = oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab)
    assert np.array_equal(out[0], packed[0].numpy()[:, :cfg.nsamps].astype(np.int64).sum(axis=0))


# ----------------------------------------------------------------------------- P5
@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_p5_impulse_response(nbits):
    """A single non-zero sample a[c*][tau] = v appears at out[d][tau - delay[d][c*]] and nowhere else."""
    nchans, nsamps, ndm, maxdelay = 9, 64, 5, 23
    rng = np.random.default_rng(100 + nbits)
    delays = rng.integers(0, maxdelay + 1, size=(ndm, nchans)).astype(np.int64)
    per = 8 // nbits
    a_len = -(-(nsamps + maxdelay) // (16 * per)) * (16 * per)
    vmax = (1 << nbits) - 1
    for cstar in range(nchans):
        for tau in range(0, nsamps + maxdelay, 7):
            a = np.zeros((nchans, a_len), np.uint8)
            a[cstar, tau] = vmax
            packed = W.pack_rows(torch.from_numpy(a), nbits).numpy()
            out = oracle.dedisperse(packed, nbits, nsamps, delays)
            expect = np.zeros((ndm, nsamps), np.uint32)
            for d in range(ndm):
                t = tau - delays[d, cstar]
                if 0 <= t < nsamps:
                    expect[d, t] = vmax
            assert np.array_equal(out, expect), (cstar, tau)


# ----------------------------------------------------------------------------- P6
@pytest.mark.parametrize("nbits", [4, 8])
def test_p6_linearity(nbits):
    nchans, nsamps, ndm, maxdelay = 21, 500, 6, 40
    half = (1 << nbits) // 2
    rng = np.random.default_rng(7)
    delays = rng.integers(0, maxdelay + 1, size=(ndm, nchans)).astype(np.int64)
    per = 8 // nbits
    a_len = -(-(nsamps + maxdelay) // (16 * per)) * (16 * per)
    A = rng.integers(0, half, size=(nchans, a_len)).astype(np.uint8)
    B = rng.integers(0, half, size=(nchans, a_len)).astype(np.uint8)
    pk = lambda x: W.pack_rows(torch.from_numpy(x), nbits).numpy()
    D = lambda x: oracle.dedisperse(pk(x), nbits, nsamps, delays).astype(np.int64)
    assert np.array_equal(D(A + B), D(A) + D(B))
    assert np.array_equal(D((2 * (A // 2)).astype(np.uint8)), 2 * D(A // 2))


# ----------------------------------------------------------------------------- P7
def test_p7_time_shift():
    nbits, nchans, nsamps, ndm, maxdelay, s = 8, 13, 400, 4, 31, 17
    a, packed, delays = _random_case(nbits, nchans, nsamps + s, ndm, maxdelay, seed=77)
    full = oracle.dedisperse(packed, nbits, nsamps + s, delays)
    shifted = np.zeros_like(a)
    shifted[:, :a.shape[1] - s] = a[:, s:]
    out_shift = oracle.dedisperse(shifted, nbits, nsamps, delays)
    assert np.array_equal(out_shift, full[:, s:s + nsamps])


# ----------------------------------------------------------------------------- P8
def test_p8_injected_pulse_cfg1():
    cfg = W.CONFIGS[1]
    tab = _table(cfg)
    pulses = W.make_pulses(cfg, lambda idx: tab[idx])
    assert pulses.dm_index[0] == 10 and abs(cfg.dm_list()[10] - 50.0) < 1e-12
    packed, _ = W.gen_packed(cfg, int(tab.max()), pulses)
    out = oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab)
    d, t = np.unravel_index(np.argmax(out), out.shape)
    assert (d, t) == (10, int(pulses.t0[0]))
    # peak ~ 64*128 + 64*40 = 10752 against noise sigma 16*sqrt(64) = 128
    assert abs(int(out[d, t]) - 10752) < 6 * 128
    assert out[d, t] - np.partition(out.ravel(), -2)[-2] > 0


def test_p8_injected_pulses_cfg3_reduced():
    cfg = W.CONFIGS[3].reduced(nsamps=6000, ndm=48, nchans=512)
    tab = _table(cfg)
    pulses = W.make_pulses(cfg, lambda idx: tab[idx])
    packed, _ = W.gen_packed(cfg, int(tab.max()), pulses)
    out = oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab).astype(np.int64)
    mean = out.mean()
    for d_i, t_i in zip(pulses.dm_index, pulses.t0):
        col = out[:, t_i]
        assert col[d_i] == col.max()
        assert out[d_i, t_i] - mean >= 0.9 * cfg.pulse_amp * cfg.nchans


# ----------------------------------------------------------------------------- P9
@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_p9_three_formulations_agree(nbits):
    nchans, nsamps, ndm, maxdelay = 16, 256, 8, 45
    a, packed, delays = _random_case(nbits, nchans, nsamps, ndm, maxdelay, seed=900 + nbits)
    c_out = oracle.dedisperse(packed, nbits, nsamps, delays)
    assert np.array_equal(oracle.unpack(packed, nbits, a.shape[1]), a)
    assert np.array_equal(oracle.unpack_np(packed, nbits, a.shape[1]), a)
    assert np.array_equal(c_out, oracle.dedisperse_gather_np(a, delays, nsamps))
    assert np.array_equal(c_out[:3, :40], np.asarray(oracle.dedisperse_loops_py(a, delays[:3], 40)))
    # per-point evaluation agrees too
    rng = np.random.default_rng(1)
    d_idx, t_idx = rng.integers(0, ndm, 50), rng.integers(0, nsamps, 50)
    pts = oracle.dedisperse_points(lambda c, t: a[c, t], delays, d_idx, t_idx)
    assert np.array_equal(pts, c_out[d_idx, t_idx])
    # threads do not change the answer
    assert np.array_equal(c_out, oracle.dedisperse(packed, nbits, nsamps, delays, nthreads=1))


def test_p9_hand_worked_transform(golden_dir):
    spec = {"delay": [], "in": [], "out": []}
    for row in _read_rows(os.path.join(golden_dir, "tiny_transform.txt")):
        if row[0] in spec:
            spec[row[0]].append([int(x) for x in row[1:]])
    a = np.zeros((3, 16), np.uint8)
    a[:, :7] = np.asarray(spec["in"], np.uint8)
    delays = np.asarray(spec["delay"], np.int64)
    expect = np.asarray(spec["out"], np.uint32)
    for nbits in (2, 4, 8):
        packed = np.zeros((3, 16), np.uint8)
        pk = W.pack_rows(torch.from_numpy(a), nbits).numpy()
        packed[:, :pk.shape[1]] = pk
        assert np.array_equal(oracle.dedisperse(packed, nbits, 4, delays), expect)
    assert np.array_equal(oracle.dedisperse_gather_np(a, delays, 4), expect)


# ---------------------------------------------------------------------------- P10
def test_p10_statistics_cfg2_reduced():
    cfg = W.CONFIGS[2].reduced(nsamps=4096, ndm=16)
    tab = _table(cfg)
    packed, _ = W.gen_packed(cfg, int(tab.max()))
    out = oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab).astype(np.float64)
    assert out.max() <= 1024 * 3
    assert abs(out.mean() - 1536.0) < 1.0            # 1024 * 1.5
    assert abs(out.std() - math.sqrt(1024 * 1.25)) < 0.5


def test_p10_output_ranges():
    assert 1024 * 15 == 15360 < 65536          # cfg4 fits uint16
    assert 4096 * 255 == 1044480 < (1 << 24)   # cfg3 exact in float32
    with pytest.raises(AssertionError):
        oracle.cast_out(np.array([70000]), "u16")
    with pytest.raises(AssertionError):
        oracle.cast_out(np.array([1 << 24]), "f32")
    assert oracle.cast_out(np.array([16777215]), "f32")[0] == 16777215.0


# ---------------------------------------------------------------------------- P11
def test_p11_packing_convention():
    assert oracle.unpack(np.array([[0xE4]], np.uint8), 2, 4).tolist() == [[0, 1, 2, 3]]
    assert oracle.unpack(np.array([[0x21]], np.uint8), 4, 2).tolist() == [[1, 2]]
    assert oracle.unpack(np.array([[0xAB]], np.uint8), 8, 1).tolist() == [[0xAB]]
    assert W.pack_rows(torch.tensor([[0, 1, 2, 3]], dtype=torch.uint8), 2).tolist() == [[0xE4]]
    assert W.pack_rows(torch.tensor([[1, 2]], dtype=torch.uint8), 4).tolist() == [[0x21]]
    rng = np.random.default_rng(5)
    for nbits in (2, 4, 8):
        a = rng.integers(0, 1 << nbits, size=(3, 64)).astype(np.uint8)
        p = W.pack_rows(torch.from_numpy(a), nbits).numpy()
        assert p.shape == (3, 64 * nbits // 8)
        assert np.array_equal(oracle.unpack(p, nbits, 64), a)


# ----------------------------------------------------------------------------- P12
@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_p12_kill_mask(nbits):
    """`sum += data * kill_mask[channel]`.  Pinned by what the mask must mean, through paths that
    never touch the mask argument: (i) zeroing the killed rows of the INPUT and summing everything; (ii) the sum
    over the kept channels only, as a smaller problem; (iii) complementary masks add up to the unmasked sum."""
    nchans, nsamps, ndm, maxdelay = 23, 300, 6, 40
    a, packed, delays = _random_case(nbits, nchans, nsamps, ndm, maxdelay, seed=1200 + nbits)
    rng = np.random.default_rng(12)
    mask = (rng.random(nchans) < 0.6).astype(np.int32)
    mask[0], mask[1] = 0, 1                       # both values certainly present
    masked = oracle.dedisperse(packed, nbits, nsamps, delays, mask=mask)
    # (i) zero the killed rows, no mask
    a0 = a.copy()
    a0[mask == 0] = 0
    p0 = W.pack_rows(torch.from_numpy(a0), nbits).numpy()
    assert np.array_equal(masked, oracle.dedisperse(p0, nbits, nsamps, delays))
    # (ii) the kept channels alone
    keep = np.nonzero(mask)[0]
    assert np.array_equal(masked, oracle.dedisperse(packed[keep], nbits, nsamps, delays[:, keep]))
    # (iii) complements
    comp = oracle.dedisperse(packed, nbits, nsamps, delays, mask=1 - mask)
    full = oracle.dedisperse(packed, nbits, nsamps, delays)
    assert np.array_equal(masked.astype(np.int64) + comp, full)
    # any nonzero mask value keeps the channel; all ones == no mask; all zeros == 0
    assert np.array_equal(oracle.dedisperse(packed, nbits, nsamps, delays, mask=mask * 7), masked)
    assert np.array_equal(oracle.dedisperse(packed, nbits, nsamps, delays, mask=np.ones(nchans)), full)
    assert not oracle.dedisperse(packed, nbits, nsamps, delays, mask=np.zeros(nchans)).any()
    # the unpacked entry point and the per-point form take the same mask
    assert np.array_equal(oracle.dedisperse_unpacked(a, nsamps, delays, mask=mask), masked)
    d_idx, t_idx = rng.integers(0, ndm, 40), rng.integers(0, nsamps, 40)
    pts = oracle.dedisperse_points(lambda c, t: a[c, t], delays, d_idx, t_idx, mask=mask)
    assert np.array_equal(pts, masked[d_idx, t_idx])


# ----------------------------------------------------------------------------- P13
def _subband_case(nbits, sb, grp, seed, nchans=24, ndm=11, nsamps=200):
    cfg = W.CONFIGS[1]
    dms = np.arange(ndm, dtype=np.float64) * 7.5
    nominal, d1, d2 = oracle.subband_tables(nchans, cfg.dt, cfg.f_top, -2.0, dms, sb, grp)
    need = oracle.subband_required_samples(nsamps, d1, d2, sb)
    rng = np.random.default_rng(seed)
    per = 8 // nbits
    a_len = -(-need // (16 * per)) * (16 * per)
    a = rng.integers(0, 1 << nbits, size=(nchans, a_len)).astype(np.uint8)
    packed = W.pack_rows(torch.from_numpy(a), nbits).numpy()
    return cfg, dms, nominal, d1, d2, a, packed


@pytest.mark.parametrize("nbits", [2, 8])
def test_p13_subband_one_channel_subbands_is_the_direct_transform(nbits):
    """N'nu = 1: step 1 copies the channels (delta1 = 0) and step 2 is eq. 3, whatever N'DM is."""
    nchans, nsamps = 24, 200
    for grp in (1, 4):
        cfg, dms, nominal, d1, d2, a, packed = _subband_case(nbits, 1, grp, seed=13)
        assert not d1.any()
        exact = oracle.delay_table(nchans, cfg.dt, cfg.f_top, -2.0, dms)
        assert np.array_equal(d2, exact)
        got = oracle.subband_dedisperse(packed, nbits, nsamps, nchans, cfg.dt, cfg.f_top, -2.0, dms, 1, grp)
        assert np.array_equal(got, oracle.dedisperse(packed, nbits, nsamps, exact))


@pytest.mark.parametrize("sb,grp", [(4, 1), (4, 3), (8, 4), (24, 11)])
def test_p13_subband_equals_direct_with_summed_delays_and_error_bound(sb, grp):
    """The two steps are linear, so the result is eq. 3 with delay delta1[g(d)][c] + delta2[d][c // N'nu] (run through
    the pinned C loop); that delay differs from eq. 5 by at most 1 + |DMnom - DM| (DeltaT(c) - DeltaT(first channel of
    the sub-band)) samples -- two roundings plus the nominal-DM approximation inside the sub-band."""
    nbits, nchans, nsamps = 4, 24, 200
    cfg, dms, nominal, d1, d2, a, packed = _subband_case(nbits, sb, grp, seed=131)
    got = oracle.subband_dedisperse(packed, nbits, nsamps, nchans, cfg.dt, cfg.f_top, -2.0, dms, sb, grp)
    g_of_d = np.arange(len(dms)) // grp
    eff = d1[g_of_d] + d2[:, np.arange(nchans) // sb]
    assert np.array_equal(got, oracle.dedisperse(packed, nbits, nsamps, eff))
    # DM 0 is its own nominal DM only when it sits in the middle of its group; its row is the channel sum when grp == 1
    if grp == 1:
        assert np.array_equal(got[0], a[:, :nsamps].astype(np.int64).sum(axis=0))
    f = cfg.f_top + np.arange(nchans) * -2.0
    T = 4.148808e3 / cfg.dt * (1.0 / f ** 2 - 1.0 / cfg.f_top ** 2)
    Tsb = T[np.arange(nchans) // sb * sb]
    bound = 1.0 + np.abs(dms[nominal][g_of_d] - dms)[:, None] * (T - Tsb)[None, :]
    exact_x = dms[:, None] * T[None, :]
    assert np.all(np.abs(eff - exact_x) <= bound + 1e-9)
    assert np.abs(eff - np.floor(exact_x + 0.5)).max() >= (1 if grp > 1 else 0)    # and the approximation is real
    # masks pass through step 1
    mask = (np.arange(nchans) % 5 != 2).astype(np.int32)
    gm = oracle.subband_dedisperse(packed, nbits, nsamps, nchans, cfg.dt, cfg.f_top, -2.0, dms, sb, grp, mask=mask)
    assert np.array_equal(gm, oracle.dedisperse(packed, nbits, nsamps, eff, mask=mask))


def test_p13_subband_impulse_response():
    """One non-zero input sample a[c*][tau] shows up in trial d at t = tau - delta1 - delta2 and nowhere else."""
    nchans, nsamps, sb, grp = 12, 64, 4, 2
    cfg = W.CONFIGS[1]
    dms = np.array([0.0, 30.0, 60.0, 90.0, 120.0])
    nominal, d1, d2 = oracle.subband_tables(nchans, cfg.dt, cfg.f_top, -5.0, dms, sb, grp)
    assert nominal.tolist() == [1, 3, 4]
    need = oracle.subband_required_samples(nsamps, d1, d2, sb)
    for cstar in (0, 5, 11):
        for tau in (0, 17, need - 1):
            a = np.zeros((nchans, need), dtype=np.uint8)
            a[cstar, tau] = 3
            out = oracle.subband_dedisperse_np(a, nsamps, nominal, d1, d2, sb, grp)
            for d in range(len(dms)):
                t = tau - int(d1[d // grp][cstar]) - int(d2[d][cstar // sb])
                want = np.zeros(nsamps, dtype=np.int64)
                if 0 <= t < nsamps:
                    want[t] = 3
                assert np.array_equal(out[d], want)


@pytest.mark.parametrize("sb,grp,nchans,ndm", [(4, 1, 24, 11), (4, 3, 24, 11), (8, 4, 24, 11), (24, 11, 24, 11), (1, 4, 24, 7), (6, 2, 36, 9)])
def test_p13_subband_required_samples_is_exactly_the_largest_index_read(sb, grp, nchans, ndm):
    """S4 pinned from both sides: step 2 reads S[b][g] at t + delta2[d][b] for t < nsamps,
    step 1 makes S[b][g][t'] from a[c][t' + delta1[g][c]], c in sub-band b, for every nominal DM g.  The largest input
    index the two steps read is therefore, by brute force over every (sub-band, nominal group, trial),
    nsamps - 1 + max_d delta2[d][b] + max_{g, c in b} delta1[g][c]; `need` must be that + 1 -- an over-estimate would
    pass every other pin (and the GPU's dd_get_subband_extent is compared with this function)."""
    cfg = W.CONFIGS[1]
    nsamps = 200
    dms = np.arange(ndm, dtype=np.float64) * 7.5
    nominal, d1, d2 = oracle.subband_tables(nchans, cfg.dt, cfg.f_top, -2.0, dms, sb, grp)
    nsb, ngroups = nchans // sb, -(-ndm // grp)
    largest = -1
    for b in range(nsb):
        top2 = -1
        for d in range(ndm):
            top2 = max(top2, int(d2[d][b]))
        top1 = -1
        for g in range(ngroups):
            for c in range(b * sb, (b + 1) * sb):
                top1 = max(top1, int(d1[g][c]))
        largest = max(largest, nsamps - 1 + top2 + top1)
    need = oracle.subband_required_samples(nsamps, d1, d2, sb)
    assert need == largest + 1
    # and the index is really read: a non-zero sample there reaches an output of the step-by-step transform when the
    # trial whose delta2 is largest belongs to the nominal group whose delta1 is largest (always so on a band whose
    # delays grow with DM: the last trial, the last group)
    a = np.zeros((nchans, need), dtype=np.uint8)
    a[nchans - 1, need - 1] = 1
    out = oracle.subband_dedisperse_np(a, nsamps, nominal, d1, d2, sb, grp)
    assert out[ndm - 1][nsamps - 1] == 1 and out[:, :nsamps - 1].sum() == 0
    # one sample fewer is not enough for the step-by-step transform
    with pytest.raises(ValueError):
        oracle.subband_dedisperse_np(a[:, :need - 1], nsamps, nominal, d1, d2, sb, grp)


# ----------------------------------------------------------------------------- P14
def test_p14_time_scrunch():
    """adjacent pairs added.  Hand example: byte 0xE4 = 2-bit samples 0,1,2,3 -> sums 1, 5; totals are
    conserved; scrunching commutes with the DM = 0 channel sum; a pulse of width 2 aligned on a pair keeps its area
    in one sample."""
    assert oracle.time_scrunch(np.array([[0xE4]], np.uint8), 2, 2).tolist() == [[1, 5]]
    assert oracle.time_scrunch(np.array([[0x21, 0xFF]], np.uint8), 4, 2).tolist() == [[3, 30]]
    rng = np.random.default_rng(14)
    for nbits in (2, 4, 8):
        a = rng.integers(0, 1 << nbits, size=(5, 128)).astype(np.uint8)
        p = W.pack_rows(torch.from_numpy(a), nbits).numpy()
        s = oracle.time_scrunch(p, nbits, 64)
        assert s.shape == (5, 64) and np.array_equal(s.sum(axis=1), a.astype(np.int64).sum(axis=1))
        assert np.array_equal(s, a.reshape(5, 64, 2).astype(np.int64).sum(axis=2))
        assert np.array_equal(s.sum(axis=0), oracle.time_scrunch_np(a.astype(np.int64).sum(axis=0)[None, :], 64)[0])
        assert np.array_equal(oracle.time_scrunch(p, nbits, 10), s[:, :10])
    z = np.zeros((1, 32), np.uint8)
    z[0, 10:12] = 3
    assert oracle.time_scrunch_np(z, 16)[0].tolist() == [0] * 5 + [6] + [0] * 10


# --------------------------------------------------------------- oracle regression
def test_oracle_regression_file(golden_dir):
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(golden_dir, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    stored = {r[0]: tuple(int(x) for x in r[1:]) for r in _read_rows(os.path.join(golden_dir, "oracle_regression.txt"))}
    for name, cfg in mg.cases():
        assert mg.checksum(mg.run_case(cfg)) == stored[name], name


# ----------------------------------------------------------------------------- P15
def test_p15_diagonal_dm_is_the_unit_gradient_at_the_end_of_the_band():
    # exact rational arithmetic: at DM_diag the (unrounded) eq. 4 delays of the last two channels differ by 1 sample
    K = Fraction(4148808, 1000)
    for idx in (1, 2, 3, 4):
        cfg = W.CONFIGS[idx]
        dt, f_top, df = Fraction(cfg.dt).limit_denominator(10 ** 12), Fraction(cfg.f_top).limit_denominator(10 ** 9), \
            Fraction(cfg.df).limit_denominator(10 ** 12)
        fa, fb = f_top + (cfg.nchans - 2) * df, f_top + (cfg.nchans - 1) * df
        grad = K * (1 / (fb * fb) - 1 / (fa * fa)) / dt                      # samples per unit DM between the two
        got = oracle.diagonal_dm_np(cfg.nchans, cfg.dt, cfg.f_top, cfg.df)
        assert abs(Fraction(got) * grad - 1) < Fraction(1, 10 ** 9)
    # cfg1 by hand: 4148.808 * (1437^-2 - 1438^-2) / 64e-6 = 0.0436465...  ->  DM_diag = 22.9113
    assert oracle.diagonal_dm_np(64, 64e-6, 1500.0, -1.0) == pytest.approx(22.9113, abs=5e-5)
    assert oracle.diagonal_dm_np(1, 64e-6, 1500.0, -1.0) == float("inf")


def test_p15_factor_ranges_by_definition():
    diag = 32.5
    dms = np.array([0.0, 32.5, 65.0, 65.0001, 130.0, 130.0001, 260.0, 260.1, 520.0, 520.1, 1000.0, 5000.0])
    got = oracle.scrunch_factors_np(dms, diag, 64, 3)
    assert list(got) == [1, 1, 1, 2, 2, 4, 4, 8, 8, 16, 16, 64]            # 5000 > 64 * 32.5: capped at max_factor
    for dm, f in zip(dms, got):                                           # the definition: F diag < DM <= 2 F diag
        assert (f == 1 and dm <= 2 * diag) or (f * diag < dm and (dm <= 2 * f * diag or f == 64))
    assert list(oracle.scrunch_factors_np(dms, diag, 4, 3)) == [1, 1, 1, 2, 2, 4, 4, 4, 4, 4, 4, 4]
    assert list(oracle.scrunch_factors_np(dms, diag, 64, 15)) == [1, 1, 1, 2, 2, 4, 4, 8, 8, 16, 16, 16]   # 32 * 15 > 255
    assert set(oracle.scrunch_factors_np(dms, diag, 64, 255)) == {1}                                       # 8-bit input


@pytest.mark.parametrize("nbits", [2, 4])
def test_p15_levels_equal_the_full_resolution_loop_summed_over_f_outputs(nbits):
    # A_F[c][t + d] = sum_{i<F} A[c][F (t + d) + i]  =>  D_F[d][t] = sum_{i<F} D'[d][F t + i], D' = eq. 3 at full
    # resolution with the delays F * delay_F -- evaluated by the pinned C loop
    base = W.CONFIGS[2 if nbits == 2 else 4]
    nchans, nsamps = 48, 640
    dms = np.array([0.0, 40.0, 100.0, 170.0, 200.0, 390.0, 500.0, 800.0, 1500.0, 1999.0])
    diag = oracle.diagonal_dm_np(nchans, base.dt, base.f_top, base.df)
    fac = oracle.scrunch_factors_np(dms, diag, 64, (1 << nbits) - 1)
    assert len(set(fac)) >= 4 and fac[0] == 1
    need = max(int(F) * (nsamps // int(F) + int(oracle.delay_table(nchans, base.dt * int(F), base.f_top, base.df, dms[fac == F]).max()))
               for F in set(fac)) + 64
    rng = np.random.default_rng(150 + nbits)
    a = rng.integers(0, 1 << nbits, size=(nchans, need), dtype=np.int64)
    levels = oracle.scrunched_dedisperse_np(a, nsamps, nchans, base.dt, base.f_top, base.df, dms, 64, (1 << nbits) - 1)
    assert [F for F, _, _ in levels] == sorted(set(int(f) for f in fac))
    for F, first, res in levels:
        idx = np.nonzero(fac == F)[0]
        assert first == idx[0] and res.shape == (len(idx), nsamps // F)
        dF = oracle.delay_table(nchans, base.dt * F, base.f_top, base.df, dms[idx])
        full = oracle.dedisperse_unpacked(a, (nsamps // F) * F, dF * F)
        assert np.array_equal(res, full.reshape(len(idx), nsamps // F, F).sum(axis=2))
    # kill mask: the masked transform is the transform of the input with the killed rows zeroed
    mask = (np.arange(nchans) % 5 != 2).astype(np.int32)
    masked = oracle.scrunched_dedisperse_np(a, nsamps, nchans, base.dt, base.f_top, base.df, dms, 64, (1 << nbits) - 1, mask=mask)
    zeroed = oracle.scrunched_dedisperse_np(a * mask[:, None], nsamps, nchans, base.dt, base.f_top, base.df, dms, 64, (1 << nbits) - 1)
    assert all(np.array_equal(m[2], z[2]) and m[0] == z[0] for m, z in zip(masked, zeroed)) and len(masked) == len(levels)
    assert not np.array_equal(masked[0][2], levels[0][2])
    # max_factor = 1: one level, the plain transform
    one = oracle.scrunched_dedisperse_np(a, nsamps, nchans, base.dt, base.f_top, base.df, dms[:5], 1, (1 << nbits) - 1)
    assert len(one) == 1 and one[0][0] == 1
    assert np.array_equal(one[0][2], oracle.dedisperse_unpacked(a, nsamps, oracle.delay_table(nchans, base.dt, base.f_top, base.df, dms[:5])))


# ----------------------------------------------------------------------------- P16: tree dedispersion
def test_p16_theta_phi_hand_values_and_four_channel_tree():
    """Eq. 14-15 as printed, worked by hand for N = 4: step 0 (r = 1) pairs the channels as they stand with delays 0 / 1,
    step 1 (r = 2) takes Phi(2, .) = 0, 2, 1, 3 and Theta(1, .) = 0, 1, 1, 2 -- which gives the delays of eq. 8,
    round(d' nu / 3): d' = 1: 0 0 1 1, d' = 2: 0 1 1 2, d' = 3: 0 1 2 3."""
    assert [oracle.tree_phi(1, v) for v in range(4)] == [0, 1, 2, 3]
    assert [oracle.tree_theta(0, v) for v in range(4)] == [0, 1, 0, 1]
    assert [oracle.tree_phi(2, v) for v in range(4)] == [0, 2, 1, 3]
    assert [oracle.tree_theta(1, v) for v in range(4)] == [0, 1, 1, 2]
    assert oracle.tree_delays_np(4).tolist() == [[0, 0, 0, 0], [0, 0, 1, 1], [0, 1, 1, 2], [0, 1, 2, 3]]
    # N = 2 by hand: D'_0 = A0 + A1, D'_1[t] = A0[t] + A1[t + 1]
    a = np.array([[1, 2, 3, 9], [4, 5, 6, 7]])
    assert oracle.tree_np(a, 3).tolist() == [[5, 7, 9], [6, 8, 10]]


@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64, 128])
def test_p16_tree_delays_are_linear_trails(n):
    """"the delay function is now a linear function of nu that ranges from 0 to exactly d' across the
    band" -- every output holds every channel once (asserted inside), the delays start at 0, end at d', never decrease,
    equal eq. 8's round(d' nu / (N - 1)) exactly for N <= 8 and within one sample beyond (reading X1)."""
    dl = oracle.tree_delays_np(n)
    nu = np.arange(n)
    for dp in range(n):
        assert dl[dp, 0] == 0 and dl[dp, n - 1] == dp and (np.diff(dl[dp]) >= 0).all()
        eq8 = np.floor(dp * nu / (n - 1) + 0.5) if n > 1 else np.zeros(n)
        assert np.abs(dl[dp] - eq8).max() <= (0 if n <= 8 else 1)


@pytest.mark.parametrize("n,nbits", [(4, 8), (8, 2), (32, 4), (64, 8)])
def test_p16_tree_equals_the_direct_sum_with_its_delays(n, nbits):
    """Eq. 7: the tree's output IS a shifted channel sum; run through the pinned C loop (eq. 3) with the tree's delay table
    -- for N <= 8 that table is eq. 8 itself, written out here by its formula."""
    nsamps = 300
    rng = np.random.default_rng(160 + n)
    a = rng.integers(0, 1 << nbits, size=(n, nsamps + n - 1)).astype(np.uint8)
    got = oracle.tree_np(a, nsamps)
    table = (np.floor(np.arange(n)[:, None] * np.arange(n)[None, :] / (n - 1) + 0.5).astype(np.int64) if n <= 8
             else oracle.tree_delays_np(n))
    assert np.array_equal(got, oracle.dedisperse_unpacked(a, nsamps, table))
    assert np.array_equal(got[0], a[:, :nsamps].astype(np.int64).sum(axis=0))          # d' = 0: the channel sum
    # impulse response: one sample at (c*, tau) shows up in trial d' at t = tau - delay[d'][c*] and nowhere else
    dl = oracle.tree_delays_np(n)
    z = np.zeros_like(a)
    z[n - 2, 57 + n] = 1
    out = oracle.tree_np(z, nsamps)
    for dp in range(n):
        want = np.zeros(nsamps, dtype=np.int64)
        want[57 + n - dl[dp, n - 2]] = 1
        assert np.array_equal(out[dp], want)
    # and through the packed path
    packed = W.pack_rows(torch.from_numpy(np.pad(a, ((0, 0), (0, (-a.shape[1]) % 64)))), nbits).numpy()
    assert np.array_equal(oracle.tree(packed, nbits, nsamps), got)


# ----------------------------------------------------------------------------- P17: piecewise linear tree
def _pw_case(nbits, sb, nchans=64, ndm=9, nsamps=160, dm_top=20.0, seed=170):
    cfg = W.CONFIGS[1]
    dms = np.linspace(0.0, dm_top, ndm)
    dprime, dt2 = oracle.piecewise_tree_tables(nchans, cfg.dt, cfg.f_top, cfg.df, dms, sb)
    need = oracle.piecewise_tree_required_samples(nsamps, dprime, dt2, sb)
    rng = np.random.default_rng(seed)
    a = rng.integers(0, 1 << nbits, size=(nchans, -(-need // 64) * 64)).astype(np.uint8)
    return cfg, dms, dprime, dt2, need, a


def test_p17_piecewise_tables():
    """Eq. 20 and 23 (readings X3, X4): the stage-2 delays telescope to the direct delays (eq. 5, the pinned table) of the
    sub-bands' first channels; d'_n(d) is the rounded delay across the sub-band, checked in exact rational arithmetic."""
    from fractions import Fraction
    cfg, dms, dprime, dt2, need, a = _pw_case(8, 16)
    full = oracle.delay_table(64, cfg.dt, cfg.f_top, cfg.df, dms)
    assert np.array_equal(dt2, full[:, ::16])
    k, dt_ = Fraction(4148808, 1000), Fraction(cfg.dt)
    for d in (1, 4, 8):
        for n in range(4):
            f0, f1 = Fraction(cfg.f_top) + n * 16 * Fraction(cfg.df), Fraction(cfg.f_top) + (n + 1) * 16 * Fraction(cfg.df)
            x = Fraction(dms[d]) * k * (1 / f1 ** 2 - 1 / f0 ** 2) / dt_
            assert dprime[d][n] == (x + Fraction(1, 2)).__floor__()
    assert dprime[0].tolist() == [0, 0, 0, 0] and (np.diff(dprime, axis=0) >= 0).all()


@pytest.mark.parametrize("nbits,sb", [(8, 16), (2, 8), (4, 64), (8, 4)])
def test_p17_piecewise_tree_equals_the_direct_sum_with_its_delays_and_error_bound(nbits, sb):
    """Both stages are shifted sums, so the result is eq. 3 with delay  tree_delay[d'_n(d)][c - nu_n] + Dt''_n(d)  (run
    through the pinned C loop); that delay misses eq. 5's by at most the chord error of the linear trail inside the
    sub-band plus three roundings ("approximating the quadratic dispersion curve with a piecewise
    linear one").  N'nu = N with one sub-band is the basic tree; a trial beyond the diagonal is refused."""
    nchans, nsamps = 64, 160
    cfg, dms, dprime, dt2, need, a = _pw_case(nbits, sb, dm_top=20.0 if sb > 4 else 6.0)
    got = oracle.piecewise_tree_np(a, nsamps, dprime, dt2, sb)
    tdl = oracle.tree_delays_np(sb)
    c = np.arange(nchans)
    eff = tdl[dprime[:, c // sb], (c % sb)[None, :]] + dt2[:, c // sb]
    assert np.array_equal(got, oracle.dedisperse_unpacked(a, nsamps, eff))
    f = cfg.f_top + np.arange(nchans + 1) * cfg.df
    big_t = 4.148808e3 / cfg.dt * (1.0 / f ** 2 - 1.0 / cfg.f_top ** 2)
    first = c // sb * sb
    chord = (big_t[first + sb] - big_t[first]) * (c - first) / max(sb - 1, 1)
    bound = 2.0 + np.abs(dms[:, None] * (chord - (big_t[c] - big_t[first]))[None, :])
    assert np.all(np.abs(eff - dms[:, None] * big_t[c][None, :]) <= bound + 1e-9)
    assert np.array_equal(got[0], a[:, :nsamps].astype(np.int64).sum(axis=0))          # DM 0: the channel sum
    if sb == 64:      # one sub-band: stage 2 only picks the row d'_0(d) of the basic tree
        assert np.array_equal(got, oracle.tree_np(a[:, :nsamps + int(dt2.max()) + 63], nsamps)[dprime[:, 0]])
    # packed path, and the diagonal limit (reading X5)
    packed = W.pack_rows(torch.from_numpy(a), nbits).numpy()
    assert np.array_equal(oracle.piecewise_tree(packed, nbits, nsamps, nchans, cfg.dt, cfg.f_top, cfg.df, dms, sb), got)
    with pytest.raises(ValueError):
        far, far2 = oracle.piecewise_tree_tables(nchans, cfg.dt, cfg.f_top, cfg.df, [400.0], sb)
        oracle.piecewise_tree_np(np.zeros((nchans, 100000), np.uint8), nsamps, far, far2, sb)


# ------------------------------------------------------------------ P18: the frequency-padded tree
def test_p18_padding_map_hand_values():
    """Eq. 25 by hand for nu0 = 1000, dnu = -100, four channels: x = -5 (1 - (1 - 0.1 nu)^-2) = 0, 1.1728, 2.8125, 5.2041
    and 8.8889 at nu = 4: rows 0, 1, 3, 5 of a band of 9 -> 16 rows."""
    from oracle.oracle_np import padded_tree_map
    pos, npad = padded_tree_map(4, 1000.0, -100.0)
    assert pos.tolist() == [0, 1, 3, 5] and npad == 16
    pos, npad = padded_tree_map(2, 1000.0, -1e-6)          # a band so narrow that nothing stretches
    assert pos.tolist() == [0, 1] and npad == 2


@pytest.mark.parametrize("idx", [2, 3, 4])
def test_p18_padding_map_exact_and_linearising(idx):
    """Eq. 25 in exact rational arithmetic; the real channels keep their order and never share a row; N_pad is the power
    of two above nu'(N_nu) and at most twice the channel count; and the map does what eq. 24 wants: the
    quadratic delay DeltaT(nu) (eq. 4, the pinned delay table's formula) equals s nu' within half a row, s = dDeltaT/dnu at 0."""
    from fractions import Fraction
    from oracle.oracle_np import K_DM, padded_tree_map
    cfg = W.CONFIGS[idx]
    pos, npad = padded_tree_map(cfg.nchans, cfg.f_top, cfg.df)
    f0, d = Fraction(cfg.f_top), Fraction(cfg.df)
    for c in list(range(0, cfg.nchans, 37)) + [cfg.nchans - 1]:
        y = 1 + d / f0 * c
        x = Fraction(1, 2) * (f0 / d) * (1 - 1 / (y * y))
        if abs((x + Fraction(1, 2)) - round(x + Fraction(1, 2))) > Fraction(1, 10**9):     # (not within rounding noise of a tie)
            assert int(pos[c]) == (x + Fraction(1, 2)).__floor__(), c
    assert np.all(np.diff(pos) >= 1) and pos[0] == 0
    assert npad & (npad - 1) == 0 and pos[-1] < npad <= 2 * cfg.nchans and npad // 2 < pos[-1] + 2
    c = np.arange(cfg.nchans, dtype=np.float64)
    big_t = K_DM * (1.0 / (cfg.f_top + c * cfg.df) ** 2 - 1.0 / cfg.f_top ** 2) / cfg.dt                  # eq. 4
    s = K_DM / cfg.dt * (-2.0 * cfg.df / cfg.f_top ** 3)
    assert np.max(np.abs(big_t - s * pos)) <= 0.5 * s * (1 + 1e-9)


@pytest.mark.parametrize("nbits", [2, 8])
def test_p18_padded_tree_equals_the_direct_sum_with_its_delays(nbits):
    """The scatter only renames rows and blank rows add nothing: the result is eq. 3 (the pinned C loop) over the REAL
    channels with the delays of the N_pad-row tree taken at the rows eq. 25 assigns; trial 0 is the plain channel sum."""
    from oracle.oracle_np import padded_tree_map, padded_tree_np, tree_delays_np
    nchans, f_top, df, nsamps = 24, 1500.0, -8.0, 200
    pos, npad = padded_tree_map(nchans, f_top, df)
    assert npad == 32 and pos[-1] > nchans
    rng = np.random.default_rng(18 + nbits)
    a = rng.integers(0, 1 << nbits, size=(nchans, (nsamps + npad - 1 + 3) // 4 * 4), dtype=np.uint8)   # (whole bytes at 2 bits)
    got = padded_tree_np(a, nsamps, pos, npad)
    delays = tree_delays_np(npad)[:, pos]
    ref = oracle.dedisperse_unpacked(a, nsamps, delays)
    assert np.array_equal(got, ref.astype(np.int64))
    assert np.array_equal(got[0], a[:, :nsamps].astype(np.int64).sum(axis=0))
    # through the packed entry point
    packed = W.pack_rows(torch.from_numpy(a), nbits).numpy()
    rows = np.zeros((nchans, (packed.shape[1] + 15) // 16 * 16), dtype=np.uint8)
    rows[:, :packed.shape[1]] = packed
    assert np.array_equal(oracle.padded_tree(rows, nbits, nsamps, f_top, df), got)


def test_p18_trials_of_the_padded_tree():
    """Eq. 26 / X8: at DM(d') the quadratic delay of every real channel (eq. 4-5) stays within two samples and a half of
    the delay the tree applies to its row; the last trial is 1 / DeltaT(1)."""
    from oracle.oracle_np import K_DM, padded_tree_dm, padded_tree_map, tree_delays_np
    cfg = W.CONFIGS[2].reduced(nsamps=64, nchans=256)
    pos, npad = padded_tree_map(cfg.nchans, cfg.f_top, cfg.df)
    c = np.arange(cfg.nchans, dtype=np.float64)
    big_t = K_DM * (1.0 / (cfg.f_top + c * cfg.df) ** 2 - 1.0 / cfg.f_top ** 2) / cfg.dt
    dms = padded_tree_dm(np.arange(npad), npad, cfg.dt, cfg.f_top, cfg.df)
    assert dms[0] == 0 and abs(dms[-1] * big_t[1] - 1.0) < 1e-12
    tree = tree_delays_np(npad)[:, pos]
    assert np.max(np.abs(dms[:, None] * big_t[None, :] - tree)) <= 2.5
