"""dd_execute_static (include/dd.h): the entry point that allocates nothing -- kernel variant 3 with its bit-plane
work buffer in the library's fixed device array -- against the existing path (dd_execute) and the CPU oracle,
bit-exact, on two calls in a row, and with calls of other plans in between (the array is shared and keeps the last
call's contents).  Collected last on purpose (the file name sorts after the other test files).

All inputs are seeded and synthetic (dd_workloads); no expected value comes from the CUDA path other than the
existing path's output, which the parity tests pin to the oracle.
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


def _table(cfg):
    return oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.dm_list())


def _input(cfg, seed_shift=0):
    """Packed device input [nbeams][nchans][stride] of the config (another seed: other samples, same shape)."""
    c = replace(cfg, seed=cfg.seed + seed_shift)
    tab = _table(c)
    packed, stride = W.gen_packed(c, int(tab.max()), None)
    return packed, packed.cuda(), stride


def _out(cfg, kind):
    return torch.full((cfg.nbeams, cfg.ndm, cfg.nsamps), -1, dtype=_TORCH_OUT[kind], device="cuda")


def _plan(cfg):
    p = dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=3)
    p.set_dm_list(cfg.dm_list())
    return p


def _set_batch(p, cfg, packed_dev, out):
    if cfg.nbeams > 1:
        p.set_batch(cfg.nbeams, packed_dev.stride(0), out.stride(0) * out.element_size())


def _np(out, kind):
    return out.cpu().numpy().view(_NP_VIEW[kind])


# several time tiles with a ragged tail, a ragged DM block, channel counts that leave padded (all-zero) channel rows
_CASES = {
    2: dict(cfg=2, nsamps=2 * 5120 + 333, ndm=37, nchans=1000, kind="u16"),
    4: dict(cfg=4, nsamps=2 * 3072 + 77, ndm=21, nchans=250, kind="u32"),
    8: dict(cfg=5, nsamps=3072 + 501, ndm=19, nchans=123, kind="f32"),
}


def _case(nbits, nbeams=1):
    c = _CASES[nbits]
    return W.CONFIGS[c["cfg"]].reduced(nsamps=c["nsamps"], ndm=c["ndm"], nchans=c["nchans"], nbeams=nbeams), c["kind"]


@pytest.mark.parametrize("nbits", [2, 4, 8])
def test_execute_static_equals_the_existing_path_on_two_calls_in_a_row(nbits):
    cfg, kind = _case(nbits)
    stream = torch.cuda.current_stream()
    host_a, dev_a, stride = _input(cfg, 0)
    host_b, dev_b, stride_b = _input(cfg, 1000)
    assert stride == stride_b and not torch.equal(host_a, host_b)
    with _plan(cfg) as p:
        assert p.launch_info()["variant"] == 3
        want_a, want_b = _out(cfg, kind), _out(cfg, kind)
        p.execute(cfg.nsamps, dev_a, stride, want_a, _CODE[kind], stream)      # the existing path (plan-owned buffer)
        p.execute(cfg.nsamps, dev_b, stride, want_b, _CODE[kind], stream)
        got_a, got_b = _out(cfg, kind), _out(cfg, kind)
        p.execute_static(cfg.nsamps, dev_a, stride, got_a, _CODE[kind], stream)   # two calls in a row, same stream,
        p.execute_static(cfg.nsamps, dev_b, stride, got_b, _CODE[kind], stream)   # no synchronisation in between
        torch.cuda.synchronize()
        assert p.launch_info()["last_launches"] == 2
    assert np.array_equal(_np(got_a, kind), _np(want_a, kind))
    assert np.array_equal(_np(got_b, kind), _np(want_b, kind))
    assert not np.array_equal(_np(got_a, kind), _np(got_b, kind))
    ref = oracle.cast_out(oracle.dedisperse(host_a[0].numpy(), cfg.nbits, cfg.nsamps, _table(cfg)), kind)
    assert np.array_equal(_np(got_a, kind)[0], ref)


def test_execute_static_shares_one_array_between_plans_and_rewrites_what_it_reads():
    # a plan whose input is all ones in every bit leaves the array full of set bits where the next plan (other width,
    # fewer and shorter rows, padded channels) expects its all-zero rows; then back again; two beams in the last plan
    stream = torch.cuda.current_stream()
    big, _ = _case(2)
    tab_big = _table(big)
    stride_big = ((big.nsamps + int(tab_big.max())) * big.nbits // 8 + 16) // 16 * 16
    ones = torch.full((1, big.nchans, stride_big), 0xFF, dtype=torch.uint8, device="cuda")
    small, kind = _case(8, nbeams=2)
    host_s, dev_s, stride_s = _input(small)
    with _plan(big) as pb, _plan(small) as ps:
        out_big = _out(big, "u32")
        got1, got2, want = _out(small, kind), _out(small, kind), _out(small, kind)
        for o in (got1, got2, want):
            _set_batch(ps, small, dev_s, o)
        ps.execute(small.nsamps, dev_s, stride_s, want, _CODE[kind], stream)
        pb.execute_static(big.nsamps, ones, stride_big, out_big, _CODE["u32"], stream)
        ps.execute_static(small.nsamps, dev_s, stride_s, got1, _CODE[kind], stream)
        pb.execute_static(big.nsamps, ones, stride_big, out_big, _CODE["u32"], stream)
        ps.execute_static(small.nsamps, dev_s, stride_s, got2, _CODE[kind], stream)
        torch.cuda.synchronize()
        assert ps.workspace_bytes > 0 and pb.workspace_bytes == 0   # execute_static leaves the plan's own buffers alone
    assert int(_np(out_big, "u32").min()) == int(_np(out_big, "u32").max()) == 3 * big.nchans
    assert np.array_equal(_np(got1, kind), _np(want, kind))
    assert np.array_equal(_np(got2, kind), _np(want, kind))
    for b in range(small.nbeams):
        ref = oracle.cast_out(oracle.dedisperse(host_s[b].numpy(), small.nbits, small.nsamps, _table(small)), kind)
        assert np.array_equal(_np(got1, kind)[b], ref)


def test_execute_static_takes_no_device_memory():
    cfg, kind = _case(4)
    stream = torch.cuda.current_stream()
    _, dev, stride = _input(cfg)
    out = _out(cfg, kind)
    with _plan(cfg) as warm:   # loads the kernels and looks the array's address up
        warm.execute_static(cfg.nsamps, dev, stride, out, _CODE[kind], stream)
        torch.cuda.synchronize()
    with _plan(cfg) as p:      # (its tables are on the device from here on)
        torch.cuda.synchronize()
        free_before, _ = torch.cuda.mem_get_info()
        for _ in range(3):
            p.execute_static(cfg.nsamps, dev, stride, out, _CODE[kind], stream)
        torch.cuda.synchronize()
        free_after, _ = torch.cuda.mem_get_info()
        assert p.workspace_bytes == 0
    assert free_after == free_before


def test_execute_static_rejects_what_it_does_not_serve():
    stream = torch.cuda.current_stream()
    small = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    out = torch.zeros(4096, dtype=torch.int32, device="cuda")
    # beyond the array: 1024 channels of 8 bits, 70000 + delay samples per row (> 64 MiB of bit planes); the sizes are
    # checked before anything is enqueued, so the small buffers are never touched
    cfg = W.CONFIGS[5].reduced(nsamps=70000, ndm=4, nbeams=1)
    with _plan(cfg) as p:
        stride = (cfg.nsamps + p.max_delay + 15) // 16 * 16
        assert (cfg.nchans + 1) * stride > dd.DD_STATIC_WORKSPACE_BYTES
        with pytest.raises(dd.DDError) as err:
            p.execute_static(cfg.nsamps, small, stride, out, _CODE["u32"], stream)
        assert err.value.status == -11 and str(dd.DD_STATIC_WORKSPACE_BYTES) in str(err.value)
    # plans that run another kernel, or the sub-band method
    cfg, kind = _case(4)
    _, dev, stride = _input(cfg)
    o = _out(cfg, kind)
    for variant in (1, 4):
        with dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=variant) as p:
            p.set_dm_list(cfg.dm_list())
            with pytest.raises(dd.DDError) as err:
                p.execute_static(cfg.nsamps, dev, stride, o, _CODE[kind], stream)
            assert err.value.status == -12
    torch.cuda.synchronize()
    assert int(out.abs().max()) == 0 and int(_np(o, kind).min()) == int(_np(o, kind).max())   # nothing was written
