"""Second, independent formulations of the oracle in numpy / pure Python.  TEST INFRASTRUCTURE ONLY.

These exist to cross-check the C triple loop (pin P9) and to evaluate single outputs of the
full-size configs one by one (`dedisperse_points`).  They follow the paper's equations
directly (eq. 3, 4, 5) and share no code with the CUDA path.
"""
from __future__ import annotations

from typing import Callable

import numpy as np

K_DM = 4.148808e3  # MHz^2 pc^-1 cm^3 s


def delay_table_np(nchans: int, dt: float, f_top: float, df: float, dm_list) -> np.ndarray:
    """Delays in the paper's own evaluation order: the look-up table DeltaT(nu) of eq. 4
    (PAPER.md:62, 109), then eq. 5 delta_t = round(DM(d) * DeltaT(nu)), float64,
    round = floor(x + 0.5) (reading R1)."""
    nu = np.arange(nchans, dtype=np.float64)
    delta_T = (K_DM / dt) * (1.0 / (f_top + nu * df) ** 2 - 1.0 / f_top ** 2)      # eq. 4
    dm = np.asarray(dm_list, dtype=np.float64)
    return np.floor(dm[:, None] * delta_T[None, :] + 0.5).astype(np.int64)         # eq. 5


def unpack_np(packed_rows: np.ndarray, nbits: int, nsamp: int) -> np.ndarray:
    """Sample t = bits [(t*nbits)%8, +nbits) of byte (t*nbits)//8, LSB first (reading R9)."""
    p = np.asarray(packed_rows, dtype=np.uint8)
    t = np.arange(nsamp, dtype=np.int64)
    bit = t * nbits
    return ((p[..., bit // 8] >> (bit % 8).astype(np.uint8)) & ((1 << nbits) - 1)).astype(np.uint8)


def dedisperse_gather_np(a: np.ndarray, delays: np.ndarray, nsamps: int) -> np.ndarray:
    """eq. 3 as one fancy-index gather and a sum over the channel axis, per DM trial."""
    a = np.asarray(a)
    delays = np.asarray(delays, dtype=np.int64)
    nchans = a.shape[0]
    c = np.arange(nchans)[:, None]
    t = np.arange(nsamps, dtype=np.int64)[None, :]
    out = np.empty((delays.shape[0], nsamps), dtype=np.int64)
    for d in range(delays.shape[0]):
        out[d] = a[c, t + delays[d][:, None]].astype(np.int64).sum(axis=0)
    return out


def dedisperse_loops_py(a, delays, nsamps: int):
    """eq. 3 as three nested Python loops (tiny inputs only)."""
    ndm, nchans = len(delays), len(a)
    out = [[0] * nsamps for _ in range(ndm)]
    for d in range(ndm):
        for t in range(nsamps):
            s = 0
            for c in range(nchans):
                s += int(a[c][t + int(delays[d][c])])
            out[d][t] = s
    return out


def dedisperse_points(sample_fn: Callable[[np.ndarray, np.ndarray], np.ndarray], delays: np.ndarray,
                      d_idx, t_idx, mask=None) -> np.ndarray:
    """out[d_i][t_i] = sum_c sample_fn(c, t_i + delay[d_i][c]) for a list of (d_i, t_i) (eq. 3, one output at a time).

    `delays` is the full table [ndm][nchans]; `sample_fn(c, t)` returns the unpacked input values
    at integer arrays (c, t) of equal shape.  `mask` (optional, nchans values): the kill mask of PAPER.md:113,
    applied as the paper states it, by multiplication with 0 or 1.
    """
    d_idx = np.asarray(d_idx, dtype=np.int64)
    t_idx = np.asarray(t_idx, dtype=np.int64)
    rows = np.asarray(delays, dtype=np.int64)[d_idx]
    nchans = rows.shape[1]
    c = np.broadcast_to(np.arange(nchans, dtype=np.int64)[None, :], rows.shape)
    t = t_idx[:, None] + rows
    v = np.asarray(sample_fn(c, t)).astype(np.int64)
    if mask is not None:
        v = v * (np.asarray(mask) != 0).astype(np.int64)[None, :]
    return v.sum(axis=1)


# ------------------------------------------------------------------------------------------ sub-band dedispersion
# PAPER.md:317-321 (section 4.1) and 358-360 (section 4.3): "two consecutive calls to the direct dedispersion
# routine and the addition of a temporary data buffer".  The paper gives the procedure in words only; the
# readings below (S1..S4) are listed in DESIGN.md section 10.
#
#   S1  trial DMs are grouped in runs of N'DM consecutive entries of the DM list; group g covers trials
#       [g N'DM, min((g+1) N'DM, N_DM)); its nominal DM is the DM of its middle trial, index g N'DM + N'DM // 2
#       (clipped to the last trial)                          "nominal DMs, each separated by N'DM trial DMs"
#   S2  step 1 -- the direct algorithm (eq. 3) on every sub-band b of N'nu channels at every nominal DM, delays
#       by eq. 4-5 with the sub-band's first channel as the start of the band:
#           delta1[g][c] = floor(K DMnom_g (f_c^-2 - f_{b N'nu}^-2) / dt + 0.5),  b = c // N'nu
#           S[b][g][t]   = sum_{c in sub-band b} A[c][t + delta1[g][c]]
#   S3  step 2 -- the direct algorithm on the "miniature filterbank" S[.][g][.] of N_SB channels (channel b at
#       the frequency of the sub-band's first channel) for the trials of group g, delays by eq. 4-5 on the full band:
#           delta2[d][b] = floor(K DM_d (f_{b N'nu}^-2 - f_top^-2) / dt + 0.5)
#           D[d][t]      = sum_b S[b][g(d)][t + delta2[d][b]]
#   S4  step 1 is evaluated for 0 <= t < nsamps + max delta2, so the input rows must hold
#       nsamps + max_b (max delta2[.][b] + max delta1[.][sub-band b]) samples.
def subband_tables(nchans: int, dt: float, f_top: float, df: float, dm_list, sb_nchans: int, dm_group: int):
    """(nominal trial index per group [ngroups], delta1 [ngroups][nchans], delta2 [ndm][nsb]) -- S1..S3, float64."""
    dm = np.asarray(dm_list, dtype=np.float64)
    ndm = dm.shape[0]
    assert nchans % sb_nchans == 0 and dm_group >= 1
    nsb = nchans // sb_nchans
    ngroups = -(-ndm // dm_group)
    nominal = np.minimum(np.arange(ngroups) * dm_group + dm_group // 2, ndm - 1)                 # S1
    c = np.arange(nchans, dtype=np.float64)
    f = f_top + c * df
    f_sb = f_top + (np.arange(nchans) // sb_nchans * sb_nchans).astype(np.float64) * df         # first channel of c's sub-band
    delta1 = np.floor(K_DM * dm[nominal][:, None] * (1.0 / f ** 2 - 1.0 / f_sb ** 2)[None, :] / dt + 0.5).astype(np.int64)   # S2
    f_b = f_top + (np.arange(nsb) * sb_nchans).astype(np.float64) * df
    delta2 = np.floor(K_DM * dm[:, None] * (1.0 / f_b ** 2 - 1.0 / f_top ** 2)[None, :] / dt + 0.5).astype(np.int64)         # S3
    return nominal, delta1, delta2


def subband_required_samples(nsamps: int, delta1: np.ndarray, delta2: np.ndarray, sb_nchans: int) -> int:
    """S4: input samples per row the two steps read."""
    nsb = delta2.shape[1]
    d1 = delta1.reshape(delta1.shape[0], nsb, sb_nchans).max(axis=(0, 2))       # per sub-band
    return int(nsamps + (delta2.max(axis=0) + d1).max())


def subband_dedisperse_np(a: np.ndarray, nsamps: int, nominal, delta1, delta2, sb_nchans: int, dm_group: int,
                          mask=None) -> np.ndarray:
    """S2 then S3 on unpacked samples a [nchans][len]; returns int64 [ndm][nsamps].  Step by step, with the
    intermediate buffer S [nsb][ngroups][nsamps + max delta2] written out in full as the paper describes."""
    a = np.asarray(a).astype(np.int64)
    nchans = a.shape[0]
    ndm, nsb = delta2.shape
    ngroups = delta1.shape[0]
    keep = np.ones(nchans, dtype=np.int64) if mask is None else (np.asarray(mask) != 0).astype(np.int64)
    t1 = nsamps + int(delta2.max())
    S = np.zeros((nsb, ngroups, t1), dtype=np.int64)
    for b in range(nsb):                                                         # step 1 (S2)
        for g in range(ngroups):
            for c in range(b * sb_nchans, (b + 1) * sb_nchans):
                o = int(delta1[g][c])
                S[b, g] += a[c, o:o + t1] * keep[c]
    out = np.zeros((ndm, nsamps), dtype=np.int64)
    for d in range(ndm):                                                         # step 2 (S3)
        g = d // dm_group
        for b in range(nsb):
            o = int(delta2[d][b])
            out[d] += S[b, g, o:o + nsamps]
    return out


# ------------------------------------------------------------------------------------------ time-scrunching
def time_scrunch_np(a: np.ndarray, nsamps_out: int) -> np.ndarray:
    """"reduce the time resolution by a factor of two ... by adding adjacent pairs of time
    samples": out[c][t] = a[c][2t] + a[c][2t+1], 0 <= t < nsamps_out, on unpacked samples (int64 out)."""
    a = np.asarray(a).astype(np.int64)
    out = np.zeros((a.shape[0], nsamps_out), dtype=np.int64)
    for t in range(nsamps_out):
        out[:, t] = a[:, 2 * t] + a[:, 2 * t + 1]
    return out


# ------------------------------------------------------------------------------------------ scrunched transform
K_DM_SCRUNCH = 4.148808e3


def diagonal_dm_np(nchans: int, dt: float, f_top: float, df: float) -> float:
    """smearing within a channel is significant "when the gradient of a dispersion curve on the
    time-frequency grid is less than unity (i.e., beyond the 'diagonal')"; "the greatest dispersion
    delay occurs at the end of the band".  Reading T2: DM_diag = 1 / (DeltaT(nchans-1) - DeltaT(nchans-2)) with
    DeltaT(c) = k_DM (f_c^-2 - f_top^-2) / dt in samples per unit DM (eq. 4), i.e. the DM at which the last two
    channels are exactly one sample apart."""
    if nchans < 2:
        return float("inf")
    fa = f_top + (nchans - 2) * df
    fb = f_top + (nchans - 1) * df
    return 1.0 / (K_DM_SCRUNCH * (1.0 / (fb * fb) - 1.0 / (fa * fa)) / dt)


def scrunch_factors_np(dm_list, dm_diag: float, max_factor: int, vmax: int) -> np.ndarray:
    """Reading T1 (0..DM_diag and DM_diag..2 DM_diag at full resolution, then "compress time by a
    factor of 2", 2..4 DM_diag, repeat; "DMs between 2x and 4x the diagonal would proceed twice as
    fast as the computation up to 2x the diagonal"): factor 1 up to 2 DM_diag, 2^k for 2^k DM_diag < DM <= 2^(k+1)
    DM_diag.  Capped at max_factor and (reading T3) at the largest factor with factor * vmax <= 255."""
    out = []
    for dm in np.asarray(dm_list, dtype=np.float64):
        f = 1
        while f < max_factor and 2 * f * vmax <= 255 and dm > dm_diag * (2.0 * f):
            f *= 2
        out.append(f)
    return np.asarray(out, dtype=np.int64)


def scrunched_dedisperse_np(a: np.ndarray, nsamps: int, nchans: int, dt: float, f_top: float, df: float, dm_list,
                            max_factor: int, vmax: int, mask=None):
    """The direct transform with time-scrunching, step by step in the paper's order: for every
    factor F in use, the series at resolution F dt is made by adding adjacent pairs log2 F times; the trials of
    that factor are dedispersed with eq. 3-5 evaluated for the sampling interval F dt (reading T4), nsamps // F
    output samples each.  a: unpacked samples [nchans][>= needed]; mask: optional kill mask (0/1 per channel).
    -> list of (F, first trial, int64 [ndm_F][nsamps//F])."""
    dms = np.asarray(dm_list, dtype=np.float64)
    fac = scrunch_factors_np(dms, diagonal_dm_np(nchans, dt, f_top, df), max_factor, vmax)
    series = np.asarray(a).astype(np.int64)
    cur = 1
    out = []
    for F in sorted(set(int(f) for f in fac)):
        while cur < F:                                    # pairs added
            series = time_scrunch_np(series, series.shape[1] // 2)
            cur *= 2
        idx = np.nonzero(fac == F)[0]
        delays = delay_table_np(nchans, dt * F, f_top, df, dms[idx])
        ns = nsamps // F
        res = np.zeros((len(idx), ns), dtype=np.int64)
        for i in range(len(idx)):
            for c in range(nchans):
                d = int(delays[i, c])
                res[i] += series[c, d:d + ns] * (1 if mask is None else int(mask[c] != 0))
        out.append((F, int(idx[0]), res))
    return out


# ------------------------------------------------------------------------------------------ tree dedispersion
# PAPER.md:125-167 (section 3.1, eq. 7-15) and PAPER.md:181-222 (section 3.1.1, eq. 16-23).  Readings:
#   X1  The tree IS its recursion (eq. 10-13 with Theta of eq. 14 and the shuffle Phi of eq. 15 as printed; "division is
#       taken to be truncated integer division").  Eq. 7-8 describe it: the recursion's delays equal round(d' nu / (N - 1))
#       exactly for N <= 8 and deviate by at most one sample for larger N (pinned), so eq. 8 is not used to compute.
#   X2  Eq. 11-12 read: A^{i+1}[2 nu + b][t] = A^i[Phi(r, 2 nu)][t] + A^i[Phi(r, 2 nu + 1)][t + Theta(i, 2 nu + b)], r = 2^i.
#   X3  Eq. 19 (difference of two rounded delays) and eq. 20 (the difference rounded once) disagree by one sample now and
#       then; eq. 20 is taken: d'_n(d) = round(DM_d [DeltaT(nu_{n+1}) - DeltaT(nu_n)]), DeltaT(c) = k_DM (f_c^-2 - f_top^-2)/dt
#       also at c = N (one channel past the band, for the last sub-band).
#   X4  Eq. 23's sum runs over the sub-bands before n, so it telescopes: Dt''_n(d) = round(DM_d DeltaT(nu_n)) -- the direct
#       delay (eq. 5) of the sub-band's first channel.
#   X5  Eq. 16 reads N'_nu = N_nu / N_s; a trial with some d'_n(d) >= N'_nu lies beyond the diagonal DM (eq. 21) and is an
#       error of the basic method.
def tree_theta(i: int, nu: int) -> int:
    """Eq. 14: Theta(i, nu) = [(nu mod 2^(i+1)) + 1] / 2, truncated."""
    return ((nu % (1 << (i + 1))) + 1) // 2


def tree_phi(r: int, nu: int) -> int:
    """Eq. 15: Phi(r, nu) = (nu mod 2) r + nu / 2 + (nu / 2r) r, truncated divisions, r = 2^i."""
    return (nu % 2) * r + nu // 2 + (nu // (2 * r)) * r


def tree_np(a: np.ndarray, nsamps: int) -> np.ndarray:
    """Eq. 10-13 step by step on unpacked samples a [N][>= nsamps + N - 1], N a power of two: int64 D'[d'][t], d' < N,
    t < nsamps.  Samples read past the end of a row count as zero (they never reach an output t < nsamps)."""
    a = np.asarray(a).astype(np.int64)
    n = a.shape[0]
    steps = n.bit_length() - 1
    assert n == 1 << steps and a.shape[1] >= nsamps + n - 1
    length = a.shape[1]
    cur = a
    for i in range(steps):
        r = 1 << i
        nxt = np.zeros_like(cur)
        for nu in range(n // 2):
            for b in (0, 1):
                th = tree_theta(i, 2 * nu + b)
                first, second = cur[tree_phi(r, 2 * nu)], cur[tree_phi(r, 2 * nu + 1)]
                nxt[2 * nu + b] = first
                nxt[2 * nu + b, :length - th] += second[th:]
        cur = nxt
    return cur[:, :nsamps]


def tree_delays_np(n: int) -> np.ndarray:
    """The delays the recursion applies: int64 [d'][channel], found by running eq. 10-15 on index sets (every output must
    hold every channel exactly once)."""
    steps = n.bit_length() - 1
    assert n == 1 << steps
    cur = [{c: 0} for c in range(n)]
    for i in range(steps):
        r = 1 << i
        nxt = []
        for o in range(n):
            nu, th = o // 2, tree_theta(i, o)
            d = dict(cur[tree_phi(r, 2 * nu)])
            for c, dl in cur[tree_phi(r, 2 * nu + 1)].items():
                assert c not in d
                d[c] = dl + th
            nxt.append(d)
        cur = nxt
    out = np.zeros((n, n), dtype=np.int64)
    for dp in range(n):
        assert sorted(cur[dp]) == list(range(n))
        for c, dl in cur[dp].items():
            out[dp, c] = dl
    return out


def piecewise_tree_tables(nchans: int, dt: float, f_top: float, df: float, dm_list, sb_nchans: int):
    """Eq. 19-23 (readings X3, X4): (d'_n(d) [ndm][Ns], Dt''_n(d) [ndm][Ns]) for sub-bands of sb_nchans channels, float64."""
    dm = np.asarray(dm_list, dtype=np.float64)
    assert nchans % sb_nchans == 0
    ns = nchans // sb_nchans
    edges = f_top + (np.arange(ns + 1) * sb_nchans).astype(np.float64) * df          # nu_0 .. nu_Ns
    big_t = K_DM * (1.0 / edges ** 2 - 1.0 / (f_top * f_top)) / dt                  # DeltaT(nu_n), eq. 4
    dprime = np.floor(dm[:, None] * (big_t[1:] - big_t[:-1])[None, :] + 0.5).astype(np.int64)     # eq. 20
    dt2 = np.floor(dm[:, None] * big_t[:-1][None, :] + 0.5).astype(np.int64)                      # eq. 23
    return dprime, dt2


def piecewise_tree_required_samples(nsamps: int, dprime: np.ndarray, dt2: np.ndarray, sb_nchans: int) -> int:
    """Input samples per row the two stages read: stage 2 reads S_n at t + Dt''_n(d) for t < nsamps, stage 1 makes
    S_n[d'][t'] from samples up to t' + d' (the tree's delays reach d' at the sub-band's last channel); stage 1 is run on
    whole rows of nsamps + max Dt'' + sb_nchans - 1 samples."""
    return int(nsamps + dt2.max() + sb_nchans - 1)


def piecewise_tree_np(a: np.ndarray, nsamps: int, dprime: np.ndarray, dt2: np.ndarray, sb_nchans: int) -> np.ndarray:
    """Stage 1 (eq. 18: the tree on every sub-band) then stage 2 (eq. 22) on unpacked samples a [nchans][>= required];
    int64 [ndm][nsamps].  A trial beyond the diagonal (some d'_n >= sb_nchans) is an error (reading X5)."""
    a = np.asarray(a).astype(np.int64)
    nchans = a.shape[0]
    ndm, ns = dprime.shape
    assert ns * sb_nchans == nchans
    if dprime.max() >= sb_nchans:
        raise ValueError("a trial lies beyond the diagonal DM of the piecewise linear tree")
    t1 = nsamps + int(dt2.max())
    need = t1 + sb_nchans - 1
    assert a.shape[1] >= need
    s = np.zeros((ns, sb_nchans, t1), dtype=np.int64)
    for n in range(ns):                                                              # stage 1
        s[n] = tree_np(a[n * sb_nchans:(n + 1) * sb_nchans, :need], t1)
    out = np.zeros((ndm, nsamps), dtype=np.int64)
    for d in range(ndm):                                                             # stage 2
        for n in range(ns):
            o = int(dt2[d][n])
            out[d] += s[n, int(dprime[d][n]), o:o + nsamps]
    return out


# ------------------------------------------------------------------------------------------ frequency-padded tree
# PAPER.md:224-242 (section 3.1.2, eq. 24-26) and PAPER.md:307 (how the paper applies it).  Readings:
#   X6  Eq. 25 gives the row of real channel nu in the stretched band, nu' = round(x(nu)),
#       x(nu) = 1/2 (nu0 / dnu) [1 - (1 + (dnu / nu0) nu)^-2], rounded as everywhere else (floor(x + 0.5), reading R1).  x is
#       exactly DeltaT(nu) / s with s = d DeltaT / d nu at nu = 0 (eq. 24): the quadratic delays become s nu', a straight line.
#   X7  "Evaluating at nu = N_nu gives the total number of frequency channels in the linearised coordinates ... rounded up
#       to a power of two": N_pad = the smallest power of two >= nu'(N_nu).  The blank rows are zero (the
#       array is initialised to zero and the input is scattered into it) and the basic tree runs on the N_pad rows.
#   X8  The trials are those of the basic tree on the stretched band (eq. 9 with eq. 26): trial d' = N_pad - 1 is
#       DM_diag(padded) = 1 / DeltaT(1), and DM(d') = d' / ((N_pad - 1) DeltaT(1)).
def padded_tree_map(nchans: int, f_top: float, df: float):
    """Eq. 25 (X6, X7): (row of every real channel in the stretched band, int64 [nchans]; N_pad)."""
    nu = np.arange(nchans + 1, dtype=np.float64)
    y = 1.0 + (df / f_top) * nu
    x = 0.5 * (f_top / df) * (1.0 - 1.0 / (y * y))
    pos = np.floor(x + 0.5).astype(np.int64)
    npad = 1
    while npad < int(pos[nchans]):
        npad *= 2
    return pos[:nchans], npad


def padded_tree_np(a: np.ndarray, nsamps: int, pos: np.ndarray, npad: int) -> np.ndarray:
    """scatter the rows of a [nchans][>= nsamps + npad - 1] into a zero array of npad rows at pos, then the
    basic tree (eq. 10-13): int64 D'[d'][t], d' < npad."""
    a = np.asarray(a).astype(np.int64)
    assert a.shape[1] >= nsamps + npad - 1 and len(pos) == a.shape[0]
    padded = np.zeros((npad, nsamps + npad - 1), dtype=np.int64)
    for c in range(a.shape[0]):
        padded[int(pos[c])] = a[c, :nsamps + npad - 1]
    return tree_np(padded, nsamps)


def padded_tree_dm(dprime, npad: int, dt: float, f_top: float, df: float):
    """Eq. 9 on the stretched band with eq. 26 (X8): the DM of trial d'."""
    big_t1 = K_DM * (1.0 / ((f_top + df) * (f_top + df)) - 1.0 / (f_top * f_top)) / dt      # DeltaT(1), eq. 4
    return np.asarray(dprime, dtype=np.float64) / ((npad - 1) * big_t1)
