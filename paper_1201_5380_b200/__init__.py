"""paper_1201_5380_b200 -- B200-native direct incoherent dedispersion (arXiv:1201.5380, eq. 3-5).

Thin Python binding over the C ABI of `include/dd.h` (libdd_b200.so, built in-tree by
`paper_1201_5380_b200/build.py`).  The functions have the same names as the C entry points and
only marshal arguments: every step of the hot path runs in the library's CUDA kernels.  PyTorch
is used by callers for device memory and streams only.

There is NO CPU fallback.  Importing this package does not load the library; the first call
does, and raises `DDLibraryError` if the CUDA extension has not been built.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

__all__ = [
    "DDError", "DDLibraryError", "lib", "library_path",
    "dd_plan_create", "dd_plan_destroy", "dd_set_dm_list", "dd_get_delay_table", "dd_get_max_delay",
    "dd_set_batch", "dd_set_killmask", "dd_set_output_stride", "dd_set_input_max", "dd_set_subband", "dd_get_subband_extent", "dd_get_subband_tables",
    "dd_time_scrunch", "dd_execute", "dd_execute_static", "DD_STATIC_WORKSPACE_BYTES", "dd_execute_host", "dd_get_launch_info", "dd_int_add_peak",
    "dd_set_kernel_variant", "dd_set_tuning", "DD_TUNE_SUBBAND_GPC", "DD_TUNE_GROUP_SIZE", "DD_TUNE_GROUPS_PER_STAGE",
    "DD_TUNE_PAIR_TILES", "DD_TUNE_TILES_PER_CTA", "DD_TUNE_HOST_SLAB", "dd_set_workspace_limit", "dd_get_workspace_bytes", "dd_profile_enable", "dd_profile_read", "dd_strerror", "dd_last_cuda_error", "Plan",
    "dd_scrunch_create", "dd_scrunch_set_killmask", "dd_scrunch_levels", "dd_scrunch_level_info", "dd_scrunch_required_bytes", "dd_scrunch_execute",
    "dd_scrunch_destroy", "ScrunchSet",
    "dd_tree_create", "dd_tree_create_padded", "dd_tree_get_padding", "dd_tree_set_dm_list", "dd_tree_get_tables", "dd_tree_get_delays", "dd_tree_required_samples", "dd_tree_execute",
    "dd_tree_set_tuning", "dd_tree_get_info", "dd_tree_destroy", "Tree",
    "DD_OUT_F32", "DD_OUT_U16", "DD_OUT_U32", "EXPORTED_SYMBOLS",
]

DD_OUT_F32, DD_OUT_U16, DD_OUT_U32 = 32, 16, -32
DD_STATIC_WORKSPACE_BYTES = 64 * 1024 * 1024   # include/dd.h: the scratch array of dd_execute_static

# every symbol include/dd.h declares (tests check the library exports exactly these)
EXPORTED_SYMBOLS = (
    "dd_plan_create", "dd_plan_destroy", "dd_set_dm_list", "dd_get_delay_table", "dd_get_max_delay",
    "dd_set_batch", "dd_set_killmask", "dd_set_output_stride", "dd_set_input_max", "dd_set_subband", "dd_get_subband_extent", "dd_get_subband_tables",
    "dd_time_scrunch", "dd_execute", "dd_execute_static", "dd_execute_host", "dd_get_launch_info", "dd_int_add_peak",
    "dd_set_kernel_variant", "dd_set_tuning", "dd_set_workspace_limit", "dd_get_workspace_bytes", "dd_profile_enable", "dd_profile_read",
    "dd_strerror", "dd_last_cuda_error",
    "dd_scrunch_create", "dd_scrunch_set_killmask", "dd_scrunch_levels", "dd_scrunch_level_info", "dd_scrunch_required_bytes", "dd_scrunch_execute",
    "dd_scrunch_destroy",
    "dd_tree_create", "dd_tree_create_padded", "dd_tree_get_padding", "dd_tree_set_dm_list", "dd_tree_get_tables", "dd_tree_get_delays", "dd_tree_required_samples", "dd_tree_execute",
    "dd_tree_set_tuning", "dd_tree_get_info", "dd_tree_destroy",
)

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB: Optional[ctypes.CDLL] = None


class DDError(RuntimeError):
    """A dd_* call returned a negative status."""

    def __init__(self, status: int, where: str):
        self.status = status
        msg = f"{where}: {dd_strerror(status)} (status {status})"
        if status in (-9, -11, -12):
            msg += f" [{dd_last_cuda_error()}]"
        super().__init__(msg)


class DDLibraryError(ImportError):
    """libdd_b200.so is missing: build it with `python -m paper_1201_5380_b200.build`."""


def library_path() -> str:
    return os.path.join(_HERE, "libdd_b200.so")


def lib() -> ctypes.CDLL:
    """Load the C-ABI library (fails loudly when it has not been built; there is no fallback)."""
    global _LIB
    if _LIB is None:
        path = library_path()
        if not os.path.exists(path):
            raise DDLibraryError(f"{path} not found -- run `python -m paper_1201_5380_b200.build` "
                                 f"(nvcc, sm_100a). There is no CPU fallback.")
        L = ctypes.CDLL(path)
        vp, i32, i64, dbl = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double
        L.dd_plan_create.argtypes = [ctypes.POINTER(vp), i32, dbl, dbl, dbl, i32]
        L.dd_plan_destroy.argtypes = [vp]
        L.dd_set_dm_list.argtypes = [vp, vp, i32]
        L.dd_get_delay_table.argtypes = [vp, vp]
        L.dd_get_max_delay.argtypes = [vp]
        L.dd_get_max_delay.restype = i64
        L.dd_set_batch.argtypes = [vp, i32, i64, i64]
        L.dd_time_scrunch.argtypes = [i32, i64, vp, i64, i32, vp, i64, i32, vp]
        L.dd_time_scrunch.restype = i32
        L.dd_set_killmask.argtypes = [vp, vp]
        L.dd_set_subband.argtypes = [vp, i32, i32]
        L.dd_set_input_max.argtypes = [vp, i32]
        L.dd_set_output_stride.argtypes = [vp, i64]
        L.dd_set_output_stride.restype = i32
        L.dd_set_input_max.restype = i32
        L.dd_set_subband.restype = i32
        L.dd_get_subband_extent.argtypes = [vp]
        L.dd_get_subband_extent.restype = i64
        L.dd_get_subband_tables.argtypes = [vp, vp, vp, vp]
        L.dd_get_subband_tables.restype = i32
        L.dd_execute.argtypes = [vp, i64, vp, i64, vp, i32, vp]
        L.dd_execute_static.argtypes = [vp, i64, vp, i64, vp, i32, vp]
        L.dd_execute_host.argtypes = [vp, i64, vp, i64, vp, i32]
        L.dd_get_launch_info.argtypes = [vp, vp]
        L.dd_set_kernel_variant.argtypes = [vp, i32]
        L.dd_set_tuning.argtypes = [vp, i32, i32]
        L.dd_set_tuning.restype = i32
        L.dd_set_workspace_limit.argtypes = [vp, i64]
        L.dd_set_workspace_limit.restype = i32
        L.dd_get_workspace_bytes.argtypes = [vp]
        L.dd_get_workspace_bytes.restype = i64
        L.dd_int_add_peak.argtypes = [i32, ctypes.POINTER(dbl), vp]
        L.dd_profile_enable.argtypes = [vp, i32]
        L.dd_profile_read.argtypes = [vp, ctypes.POINTER(i32), vp, vp]
        L.dd_scrunch_create.argtypes = [ctypes.POINTER(vp), i32, dbl, dbl, dbl, i32, vp, i32, i32]
        L.dd_scrunch_levels.argtypes = [vp]
        L.dd_scrunch_set_killmask.argtypes = [vp, vp]
        L.dd_scrunch_set_killmask.restype = i32
        L.dd_scrunch_level_info.argtypes = [vp, i32, vp]
        L.dd_scrunch_required_bytes.argtypes = [vp, i64]
        L.dd_scrunch_required_bytes.restype = i64
        L.dd_scrunch_execute.argtypes = [vp, i64, vp, i64, vp, i32, vp]
        L.dd_scrunch_destroy.argtypes = [vp]
        L.dd_tree_create.argtypes = [ctypes.POINTER(vp), i32, i32, i32]
        L.dd_tree_set_dm_list.argtypes = [vp, dbl, dbl, dbl, vp, i32]
        L.dd_tree_create_padded.argtypes = [ctypes.POINTER(vp), i32, dbl, dbl, i32]
        L.dd_tree_create_padded.restype = i32
        L.dd_tree_get_padding.argtypes = [vp, vp]
        L.dd_tree_get_padding.restype = i32
        L.dd_tree_get_tables.argtypes = [vp, vp, vp]
        L.dd_tree_get_delays.argtypes = [vp, vp]
        L.dd_tree_required_samples.argtypes = [vp, i64]
        L.dd_tree_required_samples.restype = i64
        L.dd_tree_execute.argtypes = [vp, i64, vp, i64, vp, i32, vp]
        L.dd_tree_set_tuning.argtypes = [vp, i32, i32]
        L.dd_tree_get_info.argtypes = [vp, vp]
        L.dd_tree_destroy.argtypes = [vp]
        for f in (L.dd_tree_create, L.dd_tree_set_dm_list, L.dd_tree_get_tables, L.dd_tree_get_delays, L.dd_tree_execute,
                  L.dd_tree_set_tuning, L.dd_tree_get_info, L.dd_tree_destroy):
            f.restype = i32
        for name in ("dd_scrunch_create", "dd_scrunch_set_killmask", "dd_scrunch_levels", "dd_scrunch_level_info", "dd_scrunch_execute", "dd_scrunch_destroy"):
            getattr(L, name).restype = i32
        L.dd_strerror.argtypes = [i32]
        L.dd_strerror.restype = ctypes.c_char_p
        L.dd_last_cuda_error.argtypes = []
        L.dd_last_cuda_error.restype = ctypes.c_char_p
        for name in ("dd_plan_create", "dd_plan_destroy", "dd_set_dm_list", "dd_get_delay_table", "dd_set_batch",
                     "dd_set_killmask", "dd_execute", "dd_execute_host", "dd_get_launch_info", "dd_int_add_peak", "dd_set_kernel_variant",
                     "dd_profile_enable", "dd_profile_read"):
            getattr(L, name).restype = i32
        _LIB = L
    return _LIB


def _addr(x) -> int:
    """Address of a buffer: int, torch tensor (host or device), numpy array or None."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if isinstance(x, np.ndarray):
        return int(x.ctypes.data)
    raise TypeError(f"cannot take the address of {type(x)}")


def _stream(stream) -> int:
    if stream is None:
        return 0
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)          # torch.cuda.Stream


def _check(status: int, where: str) -> int:
    if status < 0:
        raise DDError(status, where)
    return status


def dd_strerror(status: int) -> str:
    return lib().dd_strerror(int(status)).decode()


def dd_last_cuda_error() -> str:
    return lib().dd_last_cuda_error().decode()


def dd_plan_create(nchans: int, dt: float, f_top: float, df: float, nbits: int) -> int:
    """-> opaque plan handle (int).  See include/dd.h."""
    h = ctypes.c_void_p()
    _check(lib().dd_plan_create(ctypes.byref(h), int(nchans), float(dt), float(f_top), float(df), int(nbits)),
           "dd_plan_create")
    return int(h.value)


def dd_plan_destroy(plan: int) -> None:
    _check(lib().dd_plan_destroy(plan), "dd_plan_destroy")


def dd_set_dm_list(plan: int, dm_list: Sequence[float]) -> None:
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    _check(lib().dd_set_dm_list(plan, dm.ctypes.data, int(dm.shape[0])), "dd_set_dm_list")


def dd_get_max_delay(plan: int) -> int:
    return _check(int(lib().dd_get_max_delay(plan)), "dd_get_max_delay")


def dd_get_delay_table(plan: int, ndm: int, nchans: int) -> np.ndarray:
    """-> int32 [ndm][nchans] (host)."""
    out = np.empty((ndm, nchans), dtype=np.int32)
    _check(lib().dd_get_delay_table(plan, out.ctypes.data), "dd_get_delay_table")
    return out


def dd_set_batch(plan: int, nbeams: int, in_beam_stride: int, out_beam_stride: int) -> None:
    _check(lib().dd_set_batch(plan, int(nbeams), int(in_beam_stride), int(out_beam_stride)), "dd_set_batch")


def dd_set_killmask(plan: int, mask) -> None:
    """mask: nchans values, nonzero = channel summed, 0 = skipped; None removes the mask."""
    if mask is None:
        _check(lib().dd_set_killmask(plan, None), "dd_set_killmask")
        return
    m = np.ascontiguousarray(np.asarray(mask) != 0, dtype=np.int32)
    _check(lib().dd_set_killmask(plan, ctypes.c_void_p(m.ctypes.data)), "dd_set_killmask")


def dd_time_scrunch(nrows: int, nsamps_out: int, in_ptr, in_stride: int, nbits_in: int, out_ptr, out_stride: int,
                    nbits_out: int, stream=None) -> None:
    """out[r][t] = in[r][2t] + in[r][2t+1] on packed DEVICE rows; asynchronous."""
    _check(lib().dd_time_scrunch(int(nrows), int(nsamps_out), _addr(in_ptr), int(in_stride), int(nbits_in), _addr(out_ptr),
                                 int(out_stride), int(nbits_out), _stream(stream)), "dd_time_scrunch")


def dd_set_output_stride(plan: int, out_dm_stride: int) -> None:
    """Bytes between the output rows of consecutive DM trials (0 = dense)."""
    _check(lib().dd_set_output_stride(plan, int(out_dm_stride)), "dd_set_output_stride")


def dd_set_input_max(plan: int, vmax: int) -> None:
    """Promise that no input sample exceeds vmax (0 withdraws it): planes that cannot be set are skipped."""
    _check(lib().dd_set_input_max(plan, int(vmax)), "dd_set_input_max")


def dd_set_subband(plan: int, sb_nchans: int, dm_group: int) -> None:
    """Sub-band method with sb_nchans channels per sub-band and dm_group trials per nominal DM;
    (0, 0) returns to the direct transform."""
    _check(lib().dd_set_subband(plan, int(sb_nchans), int(dm_group)), "dd_set_subband")


def dd_get_subband_extent(plan: int) -> int:
    r = int(lib().dd_get_subband_extent(plan))
    if r < 0:
        raise DDError(r, "dd_get_subband_extent")
    return r


def dd_get_subband_tables(plan: int, ndm: int, nchans: int, sb_nchans: int, dm_group: int):
    """(nominal [ngroups], delta1 [ngroups][nchans], delta2 [ndm][nchans // sb_nchans]) as int32 arrays."""
    ngroups = -(-ndm // dm_group)
    nominal = np.empty(ngroups, dtype=np.int32)
    d1 = np.empty((ngroups, nchans), dtype=np.int32)
    d2 = np.empty((ndm, nchans // sb_nchans), dtype=np.int32)
    _check(lib().dd_get_subband_tables(plan, ctypes.c_void_p(nominal.ctypes.data), ctypes.c_void_p(d1.ctypes.data),
                                       ctypes.c_void_p(d2.ctypes.data)), "dd_get_subband_tables")
    return nominal, d1, d2


def dd_execute(plan: int, nsamps: int, in_ptr, in_stride: int, out_ptr, out_nbits: int, stream=None) -> None:
    """Asynchronous; in_ptr/out_ptr are DEVICE buffers (tensors or addresses)."""
    _check(lib().dd_execute(plan, int(nsamps), _addr(in_ptr), int(in_stride), _addr(out_ptr), int(out_nbits),
                            _stream(stream)), "dd_execute")


def dd_execute_static(plan: int, nsamps: int, in_ptr, in_stride: int, out_ptr, out_nbits: int, stream=None) -> None:
    """dd_execute that allocates nothing: kernel variant 3 on the library's fixed scratch array (include/dd.h)."""
    _check(lib().dd_execute_static(plan, int(nsamps), _addr(in_ptr), int(in_stride), _addr(out_ptr), int(out_nbits),
                                   _stream(stream)), "dd_execute_static")


def dd_execute_host(plan: int, nsamps: int, in_host, in_stride: int, out_host, out_nbits: int) -> None:
    """Synchronous; in_host/out_host are HOST buffers (pinned tensors, numpy arrays or addresses)."""
    _check(lib().dd_execute_host(plan, int(nsamps), _addr(in_host), int(in_stride), _addr(out_host), int(out_nbits)),
           "dd_execute_host")


def dd_set_kernel_variant(plan: int, variant: int) -> None:
    """0 = automatic; takes effect at the next dd_set_dm_list."""
    _check(lib().dd_set_kernel_variant(plan, int(variant)), "dd_set_kernel_variant")


DD_TUNE_SUBBAND_GPC, DD_TUNE_GROUP_SIZE, DD_TUNE_GROUPS_PER_STAGE, DD_TUNE_PAIR_TILES, DD_TUNE_TILES_PER_CTA = 1, 2, 3, 4, 5
DD_TUNE_HOST_SLAB = 6


def dd_set_tuning(plan: int, key: int, value: int) -> None:
    """Launch-geometry knobs (include/dd.h); results never depend on them."""
    _check(lib().dd_set_tuning(plan, int(key), int(value)), "dd_set_tuning")


def dd_set_workspace_limit(plan: int, nbytes: int) -> None:
    _check(lib().dd_set_workspace_limit(plan, int(nbytes)), "dd_set_workspace_limit")


def dd_get_workspace_bytes(plan: int) -> int:
    n = int(lib().dd_get_workspace_bytes(plan))
    if n < 0:
        _check(n, "dd_get_workspace_bytes")
    return n


def dd_get_launch_info(plan: int) -> dict:
    info = np.zeros(8, dtype=np.int64)
    _check(lib().dd_get_launch_info(plan, info.ctypes.data), "dd_get_launch_info")
    keys = ("dm_block", "time_block", "chans_per_stage", "smem_bytes", "threads", "n_dm_blocks", "last_launches",
            "variant")
    return {k: int(v) for k, v in zip(keys, info)}


def dd_profile_enable(plan: int, max_executes: int) -> None:
    """Record per-kernel CUDA-event times of the next `max_executes` dd_execute calls (0 disables)."""
    _check(lib().dd_profile_enable(plan, int(max_executes)), "dd_profile_enable")


def dd_profile_read(plan: int, max_executes: int):
    """-> (prepass_ms, main_ms) float32 arrays, one entry per recorded dd_execute; synchronises; re-arms."""
    n = ctypes.c_int(0)
    pre = np.zeros(max_executes, dtype=np.float32)
    main = np.zeros(max_executes, dtype=np.float32)
    _check(lib().dd_profile_read(plan, ctypes.byref(n), pre.ctypes.data, main.ctypes.data), "dd_profile_read")
    return pre[:n.value].copy(), main[:n.value].copy()


def dd_int_add_peak(mode: int = 0, stream=None) -> float:
    """Measured 32-bit integer additions per second on the current device (synchronises)."""
    v = ctypes.c_double()
    _check(lib().dd_int_add_peak(int(mode), ctypes.byref(v), _stream(stream)), "dd_int_add_peak")
    return float(v.value)


def dd_scrunch_create(nchans: int, dt: float, f_top: float, df: float, nbits: int, dm_list: Sequence[float],
                      max_factor: int) -> int:
    """Direct transform with time-scrunching: -> opaque set handle.  See include/dd.h."""
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    h = ctypes.c_void_p()
    _check(lib().dd_scrunch_create(ctypes.byref(h), int(nchans), float(dt), float(f_top), float(df), int(nbits),
                                   dm.ctypes.data, int(dm.shape[0]), int(max_factor)), "dd_scrunch_create")
    return int(h.value)


def dd_scrunch_set_killmask(sset: int, mask) -> None:
    """Kill mask for every level of the set; None removes it."""
    if mask is None:
        _check(lib().dd_scrunch_set_killmask(sset, None), "dd_scrunch_set_killmask")
        return
    m = np.ascontiguousarray(np.asarray(mask) != 0, dtype=np.int32)
    _check(lib().dd_scrunch_set_killmask(sset, ctypes.c_void_p(m.ctypes.data)), "dd_scrunch_set_killmask")


def dd_scrunch_levels(sset: int) -> int:
    return _check(int(lib().dd_scrunch_levels(sset)), "dd_scrunch_levels")


def dd_scrunch_level_info(sset: int, level: int) -> dict:
    a = np.zeros(6, dtype=np.int64)
    _check(lib().dd_scrunch_level_info(sset, int(level), a.ctypes.data), "dd_scrunch_level_info")
    return dict(zip(("factor", "first_dm", "ndm", "max_delay", "nbits", "dm_diag_micro"), (int(v) for v in a)))


def dd_scrunch_required_bytes(sset: int, nsamps: int) -> int:
    r = int(lib().dd_scrunch_required_bytes(sset, int(nsamps)))
    if r < 0:
        raise DDError(r, "dd_scrunch_required_bytes")
    return r


def dd_scrunch_execute(sset: int, nsamps: int, in_ptr, in_stride: int, out_ptrs, out_nbits: int, stream=None) -> None:
    """out_ptrs: one DEVICE buffer per level ([ndm_l][nsamps // F_l]).  Asynchronous."""
    arr = (ctypes.c_void_p * len(out_ptrs))(*[_addr(o) for o in out_ptrs])
    _check(lib().dd_scrunch_execute(sset, int(nsamps), _addr(in_ptr), int(in_stride), arr, int(out_nbits),
                                    _stream(stream)), "dd_scrunch_execute")


def dd_scrunch_destroy(sset: int) -> None:
    _check(lib().dd_scrunch_destroy(sset), "dd_scrunch_destroy")


class ScrunchSet:
    """Context-managed handle of dd_scrunch_* (argument marshalling only)."""

    def __init__(self, nchans, dt, f_top, df, nbits, dm_list, max_factor):
        self.handle = dd_scrunch_create(nchans, dt, f_top, df, nbits, dm_list, max_factor)

    @property
    def levels(self):
        return [dd_scrunch_level_info(self.handle, l) for l in range(dd_scrunch_levels(self.handle))]

    def set_killmask(self, mask) -> "ScrunchSet":
        dd_scrunch_set_killmask(self.handle, mask)
        return self

    def required_bytes(self, nsamps: int) -> int:
        return dd_scrunch_required_bytes(self.handle, nsamps)

    def execute(self, nsamps, in_ptr, in_stride, out_ptrs, out_nbits, stream=None) -> None:
        dd_scrunch_execute(self.handle, nsamps, in_ptr, in_stride, out_ptrs, out_nbits, stream)

    def close(self) -> None:
        if self.handle:
            dd_scrunch_destroy(self.handle)
            self.handle = 0

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


# ------------------------------------------------------------------ tree / piecewise linear tree (include/dd.h: dd_tree_*)
def dd_tree_create(nchans: int, sb_nchans: int, nbits: int) -> int:
    h = ctypes.c_void_p()
    _check(lib().dd_tree_create(ctypes.byref(h), int(nchans), int(sb_nchans), int(nbits)), "dd_tree_create")
    return h.value


def dd_tree_create_padded(nchans: int, f_top: float, df: float, nbits: int) -> int:
    h = ctypes.c_void_p()
    _check(lib().dd_tree_create_padded(ctypes.byref(h), int(nchans), float(f_top), float(df), int(nbits)), "dd_tree_create_padded")
    return h.value


def dd_tree_get_padding(tree: int, nchans: int):
    """(rows of the nchans real channels in the stretched band, N_pad)."""
    pos = np.empty(nchans, dtype=np.int32)
    npad = _check(lib().dd_tree_get_padding(tree, ctypes.c_void_p(pos.ctypes.data)), "dd_tree_get_padding")
    return pos, npad


def dd_tree_destroy(tree: int) -> None:
    _check(lib().dd_tree_destroy(tree), "dd_tree_destroy")


def dd_tree_set_dm_list(tree: int, dt: float, f_top: float, df: float, dm_list: Sequence[float]) -> None:
    dm = np.ascontiguousarray(np.asarray(dm_list, dtype=np.float64))
    _check(lib().dd_tree_set_dm_list(tree, float(dt), float(f_top), float(df), ctypes.c_void_p(dm.ctypes.data), int(dm.size)),
           "dd_tree_set_dm_list")


def dd_tree_get_tables(tree: int, ndm: int, nsub: int):
    dprime = np.empty((ndm, nsub), dtype=np.int32)
    dt2 = np.empty((ndm, nsub), dtype=np.int32)
    _check(lib().dd_tree_get_tables(tree, ctypes.c_void_p(dprime.ctypes.data), ctypes.c_void_p(dt2.ctypes.data)), "dd_tree_get_tables")
    return dprime, dt2


def dd_tree_get_delays(tree: int, sb_nchans: int) -> np.ndarray:
    out = np.empty((sb_nchans, sb_nchans), dtype=np.int32)
    _check(lib().dd_tree_get_delays(tree, ctypes.c_void_p(out.ctypes.data)), "dd_tree_get_delays")
    return out


def dd_tree_required_samples(tree: int, nsamps: int) -> int:
    return _check(lib().dd_tree_required_samples(tree, int(nsamps)), "dd_tree_required_samples")


def dd_tree_execute(tree: int, nsamps: int, in_ptr, in_stride: int, out_ptr, out_nbits: int, stream=None) -> None:
    """Asynchronous; in_ptr/out_ptr are DEVICE buffers (tensors or addresses)."""
    _check(lib().dd_tree_execute(tree, int(nsamps), _addr(in_ptr), int(in_stride), _addr(out_ptr), int(out_nbits), _stream(stream)),
           "dd_tree_execute")


def dd_tree_set_tuning(tree: int, key: int, value: int) -> None:
    _check(lib().dd_tree_set_tuning(tree, int(key), int(value)), "dd_tree_set_tuning")


def dd_tree_get_info(tree: int) -> dict:
    info = (ctypes.c_int64 * 16)()
    _check(lib().dd_tree_get_info(tree, info), "dd_tree_get_info")
    n = int(info[0])
    return {"passes": n, "last_launches": int(info[1]), "device_bytes": int(info[2]),
            "steps": [int(info[3 + 2 * p]) for p in range(min(n, 6))], "tile": [int(info[4 + 2 * p]) for p in range(min(n, 6))]}


class Tree:
    """The tree transform of sub-bands of sb_nchans channels (sb_nchans == nchans: the whole band), optionally followed by
    stage 2 of the piecewise linear tree for a DM list."""

    def __init__(self, nchans: int, sb_nchans: int, nbits: int, _handle=None):
        self.nchans, self.sb_nchans, self.nbits, self.ndm = int(nchans), int(sb_nchans), int(nbits), 0
        self.handle = _handle if _handle is not None else dd_tree_create(nchans, sb_nchans, nbits)
        self.padding = None

    @classmethod
    def padded(cls, nchans: int, f_top: float, df: float, nbits: int) -> "Tree":
        """The frequency-padded tree: `nchans` is then N_pad, `padding` the rows of the real channels."""
        h = dd_tree_create_padded(nchans, f_top, df, nbits)
        pos, npad = dd_tree_get_padding(h, nchans)
        t = cls(npad, npad, nbits, _handle=h)
        t.padding = pos
        return t

    def set_dm_list(self, dt: float, f_top: float, df: float, dm_list) -> "Tree":
        dd_tree_set_dm_list(self.handle, dt, f_top, df, dm_list)
        self.ndm = len(dm_list)
        return self

    def tables(self):
        return dd_tree_get_tables(self.handle, self.ndm, self.nchans // self.sb_nchans)

    def delays(self) -> np.ndarray:
        return dd_tree_get_delays(self.handle, self.sb_nchans)

    def required_samples(self, nsamps: int) -> int:
        return dd_tree_required_samples(self.handle, nsamps)

    def set_tuning(self, key: int, value: int) -> "Tree":
        dd_tree_set_tuning(self.handle, key, value)
        return self

    def info(self) -> dict:
        return dd_tree_get_info(self.handle)

    def execute(self, nsamps, in_ptr, in_stride, out_ptr, out_nbits, stream=None) -> None:
        dd_tree_execute(self.handle, nsamps, in_ptr, in_stride, out_ptr, out_nbits, stream)

    def close(self) -> None:
        if self.handle:
            dd_tree_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Plan:
    """Owns one dd_plan handle (context manager); argument marshalling only."""

    def __init__(self, nchans: int, dt: float, f_top: float, df: float, nbits: int, variant: int = 0):
        self.nchans, self.nbits = int(nchans), int(nbits)
        self.ndm = 0
        self.handle = dd_plan_create(nchans, dt, f_top, df, nbits)
        if variant:
            dd_set_kernel_variant(self.handle, variant)

    def set_dm_list(self, dm_list) -> "Plan":
        dd_set_dm_list(self.handle, dm_list)
        self.ndm = len(dm_list)
        return self

    def set_batch(self, nbeams: int, in_beam_stride: int, out_beam_stride: int) -> "Plan":
        dd_set_batch(self.handle, nbeams, in_beam_stride, out_beam_stride)
        return self

    def set_subband(self, sb_nchans: int, dm_group: int) -> "Plan":
        dd_set_subband(self.handle, sb_nchans, dm_group)
        self._subband = (int(sb_nchans), int(dm_group))
        return self

    @property
    def subband_extent(self) -> int:
        return dd_get_subband_extent(self.handle)

    def subband_tables(self):
        sb, grp = self._subband
        return dd_get_subband_tables(self.handle, self.ndm, self.nchans, sb, grp)

    def set_output_stride(self, out_dm_stride: int) -> "Plan":
        dd_set_output_stride(self.handle, out_dm_stride)
        return self

    def set_input_max(self, vmax: int) -> "Plan":
        dd_set_input_max(self.handle, vmax)
        return self

    def set_workspace_limit(self, nbytes: int) -> "Plan":
        dd_set_workspace_limit(self.handle, nbytes)
        return self

    @property
    def workspace_bytes(self) -> int:
        return dd_get_workspace_bytes(self.handle)

    def set_tuning(self, key: int, value: int) -> "Plan":
        dd_set_tuning(self.handle, key, value)
        return self

    def set_killmask(self, mask) -> "Plan":
        if mask is not None and len(mask) != self.nchans:
            raise ValueError("kill mask must have nchans entries")
        dd_set_killmask(self.handle, mask)
        return self

    @property
    def max_delay(self) -> int:
        return dd_get_max_delay(self.handle)

    def delay_table(self) -> np.ndarray:
        return dd_get_delay_table(self.handle, self.ndm, self.nchans)

    def launch_info(self) -> dict:
        return dd_get_launch_info(self.handle)

    def execute(self, nsamps, in_ptr, in_stride, out_ptr, out_nbits, stream=None) -> None:
        dd_execute(self.handle, nsamps, in_ptr, in_stride, out_ptr, out_nbits, stream)

    def execute_static(self, nsamps, in_ptr, in_stride, out_ptr, out_nbits, stream=None) -> None:
        dd_execute_static(self.handle, nsamps, in_ptr, in_stride, out_ptr, out_nbits, stream)

    def profile_enable(self, max_executes: int) -> None:
        self._prof_cap = int(max_executes)
        dd_profile_enable(self.handle, max_executes)

    def profile_read(self):
        return dd_profile_read(self.handle, self._prof_cap)

    def execute_host(self, nsamps, in_host, in_stride, out_host, out_nbits) -> None:
        dd_execute_host(self.handle, nsamps, in_host, in_stride, out_host, out_nbits)

    def close(self) -> None:
        if self.handle:
            dd_plan_destroy(self.handle)
            self.handle = 0

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
