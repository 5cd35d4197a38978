"""lacosmic_masked_median_noalloc: step (7) for callers that cannot allocate device memory.

Who that is: code that runs inside somebody else's GPU application and is handed only its input and output buffers
(the host application owns the memory pool); a real-time loop that must not enter the CUDA allocator once it runs,
because cudaMalloc may block and synchronises the device; a process that has already spent its memory budget.  For
them the library keeps the scratch of step (7) -- five bit-planes and a counter -- in a fixed array of its own device
image (2.5 MiB per GPU, frames up to 2048 x 2048) instead of asking for a workspace.

What is checked here: the entry point gives the same bits as the existing workspace path (lacosmic_masked_median /
_bpm, which test_gpu_parity.py and test_gpu_variants.py hold against the oracle) on two calls in a row that share the
array -- the second on a different, smaller frame, so anything the first call left behind in the array would show --
and it refuses a frame beyond the limit without touching the output.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure of this side entrance
must not hide the parity tests of the main path.  It passes alone in a fresh process (where its first call does the
per-device address look-up) and after the other tests.
"""
import ctypes as C

import numpy as np
import pytest


def _rng(seed):
    return np.random.Generator(np.random.Philox(seed))


def _case(seed, shape, density, with_bpm):
    rng = _rng(seed)
    img = (rng.standard_normal(shape) * 30 + 200).astype(np.float32)
    mask = (rng.random(shape) < density).astype(np.uint8)
    if shape[0] > 8 and shape[1] > 8:
        mask[0:7, 0:7] = 1                       # pixels with no unmasked donor in their window
    bpm = (rng.random(shape) < 0.05).astype(np.uint8) if with_bpm else None
    return img, mask, bpm


@pytest.fixture(scope="module")
def lc():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    import paper_2602_17938_b200 as lc
    lc.load_library()          # raises if the CUDA library is missing: no fallback
    return lc


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_workspace_path(lc):
    import torch
    # first a frame at the limit (2048 x 2048 = 131072 bit-plane words) with a dense mask and bad pixels, then,
    # straight behind it on the same stream, a small ragged frame with a sparse mask and no bad-pixel plane:
    # the second call finds the array full of the first call's planes
    cases = [_case(7001, (2048, 2048), 0.45, True), _case(7002, (97, 203), 0.03, False),
             _case(7003, (300, 1100), 0.2, True)]
    dev = [tuple(None if a is None else torch.from_numpy(a).cuda() for a in c) for c in cases]
    outs = [torch.full(c[0].shape, float("nan"), dtype=torch.float32, device="cuda") for c in cases]
    torch.cuda.synchronize()
    for (img, mask, bpm), out in zip(dev, outs):             # back to back, no synchronisation in between
        r = lc.lacosmic_masked_median_noalloc(img, mask, out, bpm=bpm)
        assert r is out
    torch.cuda.synchronize()
    for (img, mask, bpm), out in zip(dev, outs):
        want = lc.lacosmic_masked_median(img, mask, bpm=bpm)          # the existing path, own workspace
        torch.cuda.synchronize()
        assert torch.equal(out, want), "no-alloc entry point differs from the workspace path (bit-exact is the bar)"
    # and the same frame twice gives the same answer twice
    img, mask, bpm = dev[2]
    again = torch.empty_like(outs[2])
    lc.lacosmic_masked_median_noalloc(img, mask, again, bpm=bpm)
    torch.cuda.synchronize()
    assert torch.equal(again, outs[2])


@pytest.mark.gpu
def test_frame_beyond_the_limit_is_refused_and_output_untouched(lc):
    import torch
    h, w = 2049, 2048                                            # 2049 * 64 words > 131072
    img = torch.zeros((h, w), dtype=torch.float32, device="cuda")
    mask = torch.ones((h, w), dtype=torch.uint8, device="cuda")
    out = torch.full((h, w), 5.0, dtype=torch.float32, device="cuda")
    with pytest.raises(lc.LacosmicError) as e:
        lc.lacosmic_masked_median_noalloc(img, mask, out)
    assert e.value.code == lc.ERR_TOO_LARGE and "scratch" in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 5.0).all())
    # a wide, short frame counts by words, not by pixels: 1024 x 4096 fits, 1025 x 4096 does not
    assert 1024 * lc.lacosmic_bitplane_pitch_words(4096) == lc.NOALLOC_MAX_WORDS


def test_limit_is_checked_before_any_cuda_call():
    """Runs without a GPU: the size check comes first, so the error is the library's own code, not a CUDA failure."""
    from paper_2602_17938_b200 import build, binding
    build.build()
    L = binding.load_library()
    fake = lambda a: C.c_void_p(a)                               # never dereferenced
    call = lambda h, w, i=0x10000000, o=0x30000000: L.lacosmic_masked_median_noalloc(
        fake(i), fake(0x20000000), None, fake(o), h, w, None)
    assert call(2049, 2048) == binding.ERR_TOO_LARGE
    assert call(1, 131072 * 32 + 1) == binding.ERR_TOO_LARGE
    assert call(0, 5) == -2 and call(8, 8, i=0) == -1 and call(8, 8, o=0) == -1
    assert call(8, 8, o=0x10000000) == -5
    assert b"scratch" in L.lacosmic_strerror(binding.ERR_TOO_LARGE)
