"""CPU oracle for direct incoherent dedispersion -- TEST INFRASTRUCTURE ONLY.

Plain statement of what the hot path computes, written from the paper
(arXiv:1201.5380; eq. 1, 3, 4, 5).  It is independent of the CUDA
path: nothing here imports `paper_1201_5380_b200`, and nothing there imports this.  Only
`tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import it.

Contents
  dd_oracle.c          the C triple loop (O1..O5), built by `oracle/build.py` into libdd_oracle.so
  oracle_np.py         a second, independent numpy formulation + per-point evaluation
  this file            ctypes wrapper around the C library + the O6 cast

Parity status: all functions pinned (tests/test_oracle_pins.py, pins P1..P14 in DESIGN.md §3 and §10).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

from . import build as _build
from .oracle_np import (delay_table_np, dedisperse_gather_np, dedisperse_points,  # noqa: F401
                        unpack_np, dedisperse_loops_py, subband_tables, subband_required_samples,
                        subband_dedisperse_np, time_scrunch_np, diagonal_dm_np, scrunch_factors_np,
                        scrunched_dedisperse_np, tree_theta, tree_phi, tree_np, tree_delays_np, piecewise_tree_tables,
                        piecewise_tree_required_samples, piecewise_tree_np, padded_tree_map, padded_tree_np,
                        padded_tree_dm)

_LIB: Optional[ctypes.CDLL] = None


def lib() -> ctypes.CDLL:
    """Load (building first if needed) the C oracle."""
    global _LIB
    if _LIB is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        i64, i32, dbl, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        L.oracle_delay_table.argtypes = [i32, dbl, dbl, dbl, i32, vp, vp]
        L.oracle_delay_table.restype = i32
        L.oracle_unpack_row.argtypes = [vp, i32, i64, vp]
        L.oracle_unpack_row.restype = None
        L.oracle_threads.argtypes = [i32]
        L.oracle_threads.restype = i32
        L.oracle_dedisperse_unpacked.argtypes = [i32, i64, vp, i64, i32, vp, vp, vp, i32]
        L.oracle_dedisperse_unpacked.restype = i32
        L.oracle_dedisperse.argtypes = [i32, i64, i32, vp, i64, i32, vp, vp, vp, i32]
        L.oracle_dedisperse.restype = i32
        _LIB = L
    return _LIB


def _ptr(a: np.ndarray) -> ctypes.c_void_p:
    return ctypes.c_void_p(a.ctypes.data)


def threads(nthreads: int = 0) -> int:
    """Threads the C loop will actually use for a request of `nthreads` (0 = all cores)."""
    return int(lib().oracle_threads(int(nthreads)))


def delay_table(nchans: int, dt: float, f_top: float, df: float, dm_list) -> np.ndarray:
    """O1-O3 (eq. 1, 4, 5): int64 [ndm][nchans]."""
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    out = np.empty((dm.shape[0], nchans), dtype=np.int64)
    rc = lib().oracle_delay_table(nchans, float(dt), float(f_top), float(df), dm.shape[0], _ptr(dm), _ptr(out))
    if rc != 0:
        raise ValueError(f"oracle_delay_table rc={rc}")
    return out


def unpack(packed_rows: np.ndarray, nbits: int, nsamp: int) -> np.ndarray:
    """O4: uint8 [nrows][nsamp] from packed rows uint8 [nrows][stride]."""
    p = np.ascontiguousarray(packed_rows, dtype=np.uint8)
    assert p.ndim == 2
    out = np.empty((p.shape[0], nsamp), dtype=np.uint8)
    L = lib()
    for r in range(p.shape[0]):
        L.oracle_unpack_row(ctypes.c_void_p(p[r].ctypes.data), nbits, nsamp,
                            ctypes.c_void_p(out[r].ctypes.data))
    return out


def _mask_arg(mask, nchans: int):
    """O7: None, or nchans values, nonzero = channel kept."""
    if mask is None:
        return None, None
    m = np.ascontiguousarray(np.asarray(mask) != 0, dtype=np.int32)
    assert m.shape == (nchans,)
    return m, _ptr(m)


def dedisperse(packed: np.ndarray, nbits: int, nsamps: int, delays: np.ndarray, nthreads: int = 0,
               mask=None) -> np.ndarray:
    """O4+O5 (eq. 3) for one beam: packed uint8 [nchans][stride] -> uint32 [ndm][nsamps].
    `mask` (optional): the channel kill mask of PAPER.md:113, nonzero = channel summed (O7)."""
    p = np.ascontiguousarray(packed, dtype=np.uint8)
    dl = np.ascontiguousarray(delays, dtype=np.int64)
    nchans, stride = p.shape
    assert dl.ndim == 2 and dl.shape[1] == nchans
    out = np.empty((dl.shape[0], nsamps), dtype=np.uint32)
    m, mp = _mask_arg(mask, nchans)
    rc = lib().oracle_dedisperse(nchans, nsamps, nbits, _ptr(p), stride, dl.shape[0], _ptr(dl), mp, _ptr(out),
                                 int(nthreads))
    if rc != 0:
        raise ValueError(f"oracle_dedisperse rc={rc}")
    return out


def dedisperse_unpacked(a: np.ndarray, nsamps: int, delays: np.ndarray, nthreads: int = 0, mask=None) -> np.ndarray:
    """O5 on already unpacked samples a uint8 [nchans][a_len] -> uint32 [ndm][nsamps]."""
    a = np.ascontiguousarray(a, dtype=np.uint8)
    dl = np.ascontiguousarray(delays, dtype=np.int64)
    nchans, a_len = a.shape
    assert dl.ndim == 2 and dl.shape[1] == nchans
    out = np.empty((dl.shape[0], nsamps), dtype=np.uint32)
    m, mp = _mask_arg(mask, nchans)
    rc = lib().oracle_dedisperse_unpacked(nchans, nsamps, _ptr(a), a_len, dl.shape[0], _ptr(dl), mp, _ptr(out),
                                          int(nthreads))
    if rc != 0:
        raise ValueError(f"oracle_dedisperse_unpacked rc={rc}")
    return out


def subband_dedisperse(packed: np.ndarray, nbits: int, nsamps: int, nchans: int, dt: float, f_top: float, df: float,
                       dm_list, sb_nchans: int, dm_group: int, mask=None) -> np.ndarray:
    """Sub-band dedispersion (readings S1..S4 in oracle_np.py) of one packed beam:
    uint8 [nchans][stride] -> int64 [ndm][nsamps]."""
    nominal, delta1, delta2 = subband_tables(nchans, dt, f_top, df, dm_list, sb_nchans, dm_group)
    need = subband_required_samples(nsamps, delta1, delta2, sb_nchans)
    a = unpack(packed, nbits, need)
    return subband_dedisperse_np(a, nsamps, nominal, delta1, delta2, sb_nchans, dm_group, mask=mask)


def time_scrunch(packed: np.ndarray, nbits_in: int, nsamps_out: int) -> np.ndarray:
    """Time-scrunching of packed rows uint8 [nrows][stride]: unpacked int64 sums [nrows][nsamps_out]."""
    return time_scrunch_np(unpack(packed, nbits_in, 2 * nsamps_out), nsamps_out)


def scrunched_dedisperse(packed: np.ndarray, nbits: int, nsamps: int, nchans: int, dt: float, f_top: float, df: float,
                         dm_list, max_factor: int, nsamp_in: int, mask=None):
    """Direct transform with time-scrunching of packed rows holding nsamp_in samples:
    list of (factor, first trial, int64 sums [ndm_F][nsamps // factor]).  Readings T1-T4."""
    return scrunched_dedisperse_np(unpack(packed, nbits, nsamp_in), nsamps, nchans, dt, f_top, df, dm_list, max_factor,
                                   (1 << nbits) - 1, mask=mask)


def cast_out(sums: np.ndarray, kind: str) -> np.ndarray:
    """O6: value-preserving cast of integer sums to "f32" | "u32" | "u16"; raises if a value does not fit."""
    s = np.asarray(sums)
    mx = int(s.max()) if s.size else 0
    if kind == "u32":
        assert mx < (1 << 32)
        return s.astype(np.uint32)
    if kind == "u16":
        assert mx < (1 << 16), "sum does not fit uint16"
        return s.astype(np.uint16)
    if kind == "f32":
        assert mx < (1 << 24), "sum is not exactly representable in float32"
        return s.astype(np.float32)
    raise ValueError(kind)


def tree(packed: np.ndarray, nbits: int, nsamps: int) -> np.ndarray:
    """The basic tree transform (eq. 7-15) of one packed beam uint8 [N][stride], N a power of two:
    int64 D'[d'][t], d' < N."""
    n = packed.shape[0]
    return tree_np(unpack(packed, nbits, nsamps + n - 1), nsamps)


def piecewise_tree(packed: np.ndarray, nbits: int, nsamps: int, nchans: int, dt: float, f_top: float, df: float, dm_list,
                   sb_nchans: int) -> np.ndarray:
    """The piecewise linear tree method (eq. 16-23; readings X1-X5 in oracle_np.py) of one packed beam:
    int64 [ndm][nsamps]."""
    dprime, dt2 = piecewise_tree_tables(nchans, dt, f_top, df, dm_list, sb_nchans)
    need = piecewise_tree_required_samples(nsamps, dprime, dt2, sb_nchans)
    return piecewise_tree_np(unpack(packed, nbits, need), nsamps, dprime, dt2, sb_nchans)


def padded_tree(packed: np.ndarray, nbits: int, nsamps: int, f_top: float, df: float) -> np.ndarray:
    """The frequency-padded tree (eq. 25; readings X6-X8 in oracle_np.py) of one packed beam
    uint8 [nchans][stride]: int64 D'[d'][t], d' < N_pad."""
    pos, npad = padded_tree_map(packed.shape[0], f_top, df)
    return padded_tree_np(unpack(packed, nbits, nsamps + npad - 1), nsamps, pos, npad)
