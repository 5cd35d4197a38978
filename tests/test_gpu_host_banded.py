"""The banded single-frame host path (-m gpu) against the oracle, over every pixel.

lacosmic_run_host / lacosmic_run_host_sparse copy a frame of >= 993 rows (lazy mode, gain supplied, w % 4 == 0) to the
device in eight bands on the library's copy stream and launch the first noise/S pass band by band behind the copies
(csrc/lacosmic_api.cu, run_host_frame and the `bands` branch of noise_pass).  A wrong margin or a missing wait there
makes a row of tiles read rows of the staging plane that have not arrived yet.  To make such a read visible the
staging workspace is POISONED before the call: with NaN bytes, or by running a different frame of the same shape
through it first, so stale rows never happen to hold the right pixels.  (Checked once by hand, DESIGN.md section 6:
with `upto` of the band loop raised by one row of tiles these tests fail.)

Frames: BASELINE.json configs[1] (2048 x 2048) and configs[2] (4000 x 6500, the frame of PAPER.md:31) from the seeded
generator, and narrow frames whose heights sit on the edges of the band / tile arithmetic.
"""
import numpy as np
import pytest

from paper_2602_17938_b200 import synth

pytestmark = pytest.mark.gpu

PARAMS = dict(gain=1.0, readnoise=10.0, sigclip=4.5, sigfrac=0.3, objlim=5.0, niter=4, satlevel=65535.0)


@pytest.fixture(scope="module")
def lc():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    import paper_2602_17938_b200 as lc
    lc.load_library()          # raises if the CUDA library is missing: no fallback
    return lc


def _workspace(lc, h, w, poison=0xFF):
    """Device staging workspace of the host calls, every byte `poison` (0xFF: every fp32 in it is a NaN)."""
    import torch
    ws = torch.empty(lc.lacosmic_host_workspace_bytes(h, w), dtype=torch.uint8, device="cuda")
    ws.fill_(poison)
    torch.cuda.synchronize()
    return ws


def _pin(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).pin_memory()


def _check_dense(r, o, label):
    assert np.array_equal(r["mask"].numpy(), o["mask"]), "%s: mask differs from the oracle" % label
    assert np.array_equal(r["clean"].numpy(), o["clean"]), "%s: cleaned frame differs from the oracle" % label


def _check_sparse(r, img, o, label):
    h, w = img.shape
    n = int(r["count"][0])
    assert n == int(o["mask"].sum()), "%s: count" % label
    bits = np.unpackbits(r["maskbits"].numpy().view(np.uint8), axis=1, bitorder="little")[:, :w]
    assert np.array_equal(bits, o["mask"]), "%s: bit-plane mask differs from the oracle" % label
    assert n <= r["capacity"], "%s: list truncated (%d > %d)" % (label, n, r["capacity"])
    idx, val = r["idx"].numpy()[:n], r["val"].numpy()[:n]
    assert np.array_equal(idx, np.flatnonzero(o["mask"])), "%s: index list" % label
    clean = img.copy()
    clean.flat[idx] = val
    assert np.array_equal(clean, o["clean"]), "%s: patched frame differs from the oracle" % label


# heights on both sides of the band switch (ceil(h/32) >= 32, i.e. h >= 993), one row past a tile / band boundary, a
# height whose band boundaries are not multiples of the tile height, and a tall narrow frame; widths: one TMA box
# narrower than a tile, widths that are multiples of 4 but not of 32
RAGGED = [(992, 64), (993, 64), (1000, 132), (1024, 4), (1025, 260), (1056, 36), (1999, 100), (4001, 68)]


@pytest.mark.parametrize("shape", RAGGED, ids=lambda s: "%dx%d" % s)
def test_ragged_heights_poisoned_workspace(lc, orc, shape):
    import torch
    h, w = shape
    f = synth.make_frame(h, w, seed=9000 + h, n_star=max(1, h * w // 4000), n_cr=max(1, h * w // 400), sp_frac=0.004)
    o = orc.run(f.img, **PARAMS)
    assert o["mask"].any()
    host = _pin(f.img)
    p = lc.Params(**PARAMS)
    ws = _workspace(lc, h, w)
    r = lc.lacosmic_run_host(host, p, dev_workspace=ws)
    launches = lc.lacosmic_last_launch_count()
    torch.cuda.synchronize()
    _check_dense(r, o, "dense %dx%d" % shape)
    ws.fill_(0xFF)
    torch.cuda.synchronize()
    rs = lc.lacosmic_run_host_sparse(host, p, capacity=h * w, dev_workspace=ws)
    torch.cuda.synchronize()
    _check_sparse(rs, f.img, o, "sparse %dx%d" % shape)
    # the launch sequence depends on the arguments alone: the banded path launches the first pass once per band
    # (8 launches instead of 1), so the count tells which path ran
    dev = torch.from_numpy(f.img).cuda()
    lc.lacosmic_graph_replay_enable(False)
    try:
        lc.lacosmic_run_ws(dev, p)
        direct = lc.lacosmic_last_launch_count()
    finally:
        lc.lacosmic_graph_replay_enable(True)
    torch.cuda.synchronize()
    if h >= 993:
        assert launches >= direct + 4, "the banded path did not run (%d launches, %d without bands)" % (launches, direct)
    else:
        assert launches < direct + 4


def test_config1_three_frames_back_to_back(lc, orc):
    """configs[1]: three different 2048 x 2048 frames through the SAME workspace on the same stream with no
    synchronisation in between -- each call's staging plane still holds the previous frame when its copy starts --
    dense results for the first and third, sparse for the second."""
    import torch
    frames = [synth.make_config(1, seed=s).img for s in (2, 102, 202)]
    h, w = frames[0].shape
    hosts = [_pin(f) for f in frames]
    p = lc.Params(**PARAMS)
    ws = _workspace(lc, h, w)
    r0 = lc.lacosmic_run_host(hosts[0], p, dev_workspace=ws)
    r1 = lc.lacosmic_run_host_sparse(hosts[1], p, capacity=h * w // 8, dev_workspace=ws)
    r2 = lc.lacosmic_run_host(hosts[2], p, dev_workspace=ws)
    torch.cuda.synchronize()
    outs = [orc.run(f, **PARAMS) for f in frames]
    _check_dense(r0, outs[0], "frame 0")
    _check_sparse(r1, frames[1], outs[1], "frame 1")
    _check_dense(r2, outs[2], "frame 2")
    assert not np.array_equal(outs[0]["mask"], outs[2]["mask"])


def test_config2_whole_frame_through_the_banded_path(lc, orc):
    """configs[2], the 4000 x 6500 frame the e2e figure of bench.py is quoted on: both host entry points, the workspace
    poisoned once with NaN and once with a different frame of the same shape (the same frame rotated by 180 degrees run
    through it first), every pixel against the oracle."""
    import torch
    f = synth.make_config(2)
    h, w = f.img.shape
    host = _pin(f.img)
    other = _pin(f.img[::-1, ::-1])
    p = lc.Params(**PARAMS)
    ws = _workspace(lc, h, w)
    rd = lc.lacosmic_run_host(host, p, dev_workspace=ws)                 # NaN-poisoned workspace
    torch.cuda.synchronize()
    lc.lacosmic_run_host_sparse(other, p, capacity=h * w // 16, dev_workspace=ws)   # leaves the rotated frame staged
    rs = lc.lacosmic_run_host_sparse(host, p, capacity=h * w // 16, dev_workspace=ws)
    torch.cuda.synchronize()
    ws.fill_(0xFF)
    torch.cuda.synchronize()
    rs2 = lc.lacosmic_run_host_sparse(host, p, capacity=h * w // 16, dev_workspace=ws)
    lc.lacosmic_run_host(other, p, dev_workspace=ws)
    rd2 = lc.lacosmic_run_host(host, p, dev_workspace=ws)
    torch.cuda.synchronize()
    o = orc.run(f.img, **PARAMS)
    _check_dense(rd, o, "dense, NaN-poisoned")
    _check_sparse(rs, f.img, o, "sparse, after the rotated frame")
    _check_sparse(rs2, f.img, o, "sparse, NaN-poisoned")
    _check_dense(rd2, o, "dense, after the rotated frame")
