"""The seeded input generators (dd_workloads): determinism, point evaluation, layout.  No method arithmetic here."""
import numpy as np
import torch

import dd_workloads as W


def test_hash_matches_python_bigint():
    c = torch.arange(0, 40, 7, dtype=torch.int64)[:, None]
    t = torch.tensor([0, 1, 2, 1000, 544763, (1 << 31) + 5], dtype=torch.int64)[None, :]
    for seed, beam in ((W.CONFIGS[2].seed, 0), (W.CONFIGS[5].seed, 12)):
        h = W.hash64(seed, beam, c, t)
        hb = W.hash64(seed, torch.tensor(beam), c, t)
        for i in range(c.shape[0]):
            for j in range(t.shape[1]):
                ref = W.hash64_py(seed, beam, int(c[i, 0]), int(t[0, j]))
                assert (int(h[i, j]) & ((1 << 64) - 1)) == ref
                assert int(hb[i, j]) == int(h[i, j])


def test_point_evaluation_matches_block_generation():
    for idx in (1, 2, 3, 4, 5):
        cfg = W.CONFIGS[idx]
        blk = W.gen_block(cfg, 0, 3, 9, 100, 164)
        cs = torch.tensor([3, 5, 8]); ts = torch.tensor([100, 130, 163])
        pts = W.values_at(cfg, 0, cs, ts)
        assert pts.tolist() == [int(blk[0, 0]), int(blk[2, 30]), int(blk[5, 63])]
        assert int(blk.max()) <= (1 << cfg.nbits) - 1


def test_distributions():
    g = W.gen_block(W.CONFIGS[1], 0, 0, 32, 0, 20000).double()
    assert abs(g.mean() - 128) < 0.2 and abs(g.std() - 16) < 0.2
    g3 = W.gen_block(W.CONFIGS[3], 0, 0, 32, 0, 20000).double()
    assert abs(g3.mean() - 128) < 0.2 and abs(g3.std() - 20) < 0.2
    u = W.gen_block(W.CONFIGS[2], 0, 0, 32, 0, 20000)
    cnt = torch.bincount(u.flatten().long(), minlength=4).double() / u.numel()
    assert (abs(cnt - 0.25) < 0.01).all()
    u4 = W.gen_block(W.CONFIGS[4], 0, 0, 32, 0, 20000)
    cnt = torch.bincount(u4.flatten().long(), minlength=16).double() / u4.numel()
    assert (abs(cnt - 1 / 16) < 0.005).all()
    b0 = W.gen_block(W.CONFIGS[5], 0, 0, 4, 0, 256)
    b1 = W.gen_block(W.CONFIGS[5], 1, 0, 4, 0, 256)
    assert not torch.equal(b0, b1)


def test_pulse_injection_uses_callers_tracks():
    cfg = W.CONFIGS[1]
    tracks = np.arange(cfg.nchans, dtype=np.int64)[None, :] * 2      # an arbitrary made-up track
    pulses = W.Pulses(dm_index=np.array([10]), t0=np.array([50]), tracks=tracks, amp=40)
    base = W.gen_block(cfg, 0, 0, cfg.nchans, 0, 400).to(torch.int64)
    inj = W.gen_block(cfg, 0, 0, cfg.nchans, 0, 400, pulses).to(torch.int64)
    diff = inj - base
    for c in range(cfg.nchans):
        nz = torch.nonzero(diff[c]).flatten().tolist()
        assert nz == [50 + 2 * c] and int(diff[c, 50 + 2 * c]) == 40


def test_layout_and_dm_lists():
    cfg = W.CONFIGS[2]
    nrow, stride = W.row_layout(cfg, 20476)
    assert stride == 136192 and nrow == 136192 * 4       # 544764 samples -> 136192 B
    assert W.row_layout(W.CONFIGS[3], 157502)[1] == 1206080
    assert W.row_layout(W.CONFIGS[4], 40951)[1] == 544768
    assert W.row_layout(W.CONFIGS[5], 20476)[1] == 282624
    dm1 = W.CONFIGS[1].dm_list()
    assert dm1[0] == 0 and dm1[-1] == 155 and abs(dm1[10] - 50) < 1e-12 and len(dm1) == 32
    assert W.CONFIGS[2].dm_list()[-1] == 1000.0 and W.CONFIGS[4].dm_list()[-1] == 2000.0
    r = W.CONFIGS[2].reduced(nsamps=100, ndm=10)
    assert abs(r.dm_list()[1] - W.CONFIGS[2].dm_list()[1]) < 1e-12
    packed, st = W.gen_packed(W.CONFIGS[4].reduced(nsamps=100, ndm=4, nchans=8), 30)
    assert packed.shape == (1, 8, st) and st % 16 == 0 and st * 2 >= 130
