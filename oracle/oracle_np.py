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
