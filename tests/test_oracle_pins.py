"""Pins for the CPU oracle (oracle/lacosmic_oracle.c) -- run with -m "not gpu".

Each test pins one part of the oracle to something OTHER than the oracle itself: a closed form,
a library routine whose definition coincides (scipy.ndimage), the literal 2x-grid definition of
step (1), brute force on tiny inputs, hand-computed fixtures (tests/golden/), or an invariant of
the method.  Pin numbers P1-P12 are those of SURVEY.md 8(c) / DESIGN.md section 4.
"""
import math
import os

import numpy as np
import pytest
import scipy.ndimage as ndi

from paper_2602_17938_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
PARAMS = dict(gain=1.0, readnoise=10.0, sigclip=4.5, sigfrac=0.3, objlim=5.0, niter=4,
              satlevel=65535.0)


def _rng(seed):
    return np.random.Generator(np.random.Philox(seed))


# ---------------------------------------------------------------- P1: constant image
@pytest.mark.parametrize("c", [0.0, 100.0, 1234.5, -7.0])
def test_p1_constant_image(orc, c):
    img = np.full((23, 31), c, np.float32)
    r = orc.run(img, debug_iter=0, **PARAMS)
    assert not r["Lp"].any(), "L+ must vanish everywhere including borders"
    assert not r["S"].any() and not r["Sp"].any()
    assert not r["mask"].any() and (r["counts"] == 0).all()
    assert np.array_equal(r["clean"], img)
    n = math.sqrt(1.0 * max(c, 1e-4) + 100.0) / 1.0
    assert np.allclose(r["N"], n, rtol=1e-6, atol=0)
    assert np.all(r["F"] == np.float32(0.01))


# ---------------------------------------------------------------- P2: single spike, closed form
@pytest.mark.parametrize("pos,factor", [((10, 12), 2.0), ((0, 12), 1.5), ((10, 0), 1.5),
                                        ((20, 12), 1.5), ((10, 24), 1.5), ((0, 0), 1.0),
                                        ((20, 24), 1.0), ((0, 24), 1.0), ((20, 0), 1.0)])
def test_p2_single_spike(orc, pos, factor):
    B, A = 100.0, 1000.0
    img = np.full((21, 25), B, np.float32)
    img[pos] += A
    r = orc.run(img, debug_iter=0, **PARAMS)
    lp = np.zeros_like(img)
    lp[pos] = factor * A          # interior 2A, edge 1.5A, corner A; 0 elsewhere
    assert np.array_equal(r["Lp"], lp)
    n = math.sqrt(B + 100.0)      # med5 removes the spike even in a clamped corner window
    assert np.allclose(r["N"], n, rtol=1e-6, atol=0)
    s = factor * A / (2.0 * n)    # N=14.142136 -> 70.71068 / 53.03301 / 35.35534
    assert r["S"][pos] == pytest.approx(s, rel=1e-6)
    assert np.array_equal(r["Sp"], r["S"])       # med5(S) = 0 everywhere
    assert np.all(r["m3"] == np.float32(B)) and np.all(r["F"] == np.float32(0.01))
    expect_mask = np.zeros(img.shape, np.uint8)
    expect_mask[pos] = 1
    assert np.array_equal(r["mask"], expect_mask)
    assert np.all(r["clean"] == np.float32(B))
    assert list(r["counts"]) == [1, 0, 0, 0]


def test_p2_spike_below_threshold_not_flagged(orc):
    img = np.full((21, 25), 100.0, np.float32)
    n = math.sqrt(200.0)
    img[10, 12] += np.float32(4.4 * n)           # S = A/N = 4.4 < sigclip
    r = orc.run(img, **PARAMS)
    assert not r["mask"].any()
    img[10, 12] = 100.0 + np.float32(4.6 * n)    # S = 4.6 > sigclip
    r = orc.run(img, **PARAMS)
    assert r["mask"].sum() == 1 and r["mask"][10, 12] == 1


def test_p2_laplacian_scale_is_R1(orc):
    """R1: centre weight 4, no 1/4 factor -> an isolated spike gives exactly L+ = 2A."""
    img = np.zeros((9, 9), np.float32)
    img[4, 4] = 8.0
    assert orc.lplus(img)[4, 4] == 16.0


# ---------------------------------------------------------------- O1 against the literal definition
@pytest.mark.parametrize("shape", [(1, 1), (1, 9), (7, 1), (2, 2), (17, 23)])
def test_lplus_matches_literal_2x_grid_definition(orc, shape):
    """north_star (1) written out: replicate 2x, convolve with the 3x3 Laplacian (edge-replicate on
    the 2h x 2w grid), clip negatives, 2x2 block average -- in float64 on integer-valued input,
    where every fp32 step of the oracle is exact, so equality must be exact."""
    img = _rng(7).integers(-500, 500, shape).astype(np.float32)
    big = np.kron(img.astype(np.float64), np.ones((2, 2)))
    lap = np.array([[0, -1, 0], [-1, 4, -1], [0, -1, 0]], np.float64)
    conv = ndi.convolve(big, lap, mode="nearest")
    conv[conv < 0] = 0.0
    h, w = shape
    ref = conv.reshape(h, 2, w, 2).mean(axis=(1, 3))
    assert np.array_equal(orc.lplus(img).astype(np.float64), ref)


def test_lplus_real_valued_close_to_float64_definition(orc):
    img = (_rng(8).standard_normal((40, 37)) * 30 + 100).astype(np.float32)
    big = np.kron(img.astype(np.float64), np.ones((2, 2)))
    lap = np.array([[0, -1, 0], [-1, 4, -1], [0, -1, 0]], np.float64)
    conv = np.maximum(ndi.convolve(big, lap, mode="nearest"), 0.0)
    ref = conv.reshape(40, 2, 37, 2).mean(axis=(1, 3))
    assert np.allclose(orc.lplus(img), ref, rtol=0, atol=2e-5 * np.abs(img).max())


# ---------------------------------------------------------------- P3: medians
@pytest.mark.parametrize("k", [3, 5, 7])
@pytest.mark.parametrize("shape", [(1, 1), (1, 5), (4, 1), (2, 3), (9, 9), (33, 47)])
def test_p3_median_equals_scipy_nearest(orc, k, shape):
    x = _rng(100 + k).standard_normal(shape).astype(np.float32)
    assert np.array_equal(orc.medfilt(x, k), ndi.median_filter(x, size=k, mode="nearest"))


@pytest.mark.parametrize("k", [3, 5, 7])
def test_p3_median_heavy_ties_and_plateaus(orc, k):
    rng = _rng(200 + k)
    x = rng.integers(0, 3, (40, 52)).astype(np.float32)        # three distinct values only
    x[10:20, 10:25] = 65535.0                                   # saturated plateau
    x[x == 0] = 0.0
    assert np.array_equal(orc.medfilt(x, k), ndi.median_filter(x, size=k, mode="nearest"))


@pytest.mark.parametrize("k", [3, 5, 7])
def test_p3_median_brute_force_full_sort(orc, k):
    """Independent brute force: pad by replication with numpy, full np.sort of each window."""
    rng = _rng(300 + k)
    x = rng.standard_normal((11, 13)).astype(np.float32)
    r = k // 2
    xp = np.pad(x, r, mode="edge")
    ref = np.empty_like(x)
    for y in range(x.shape[0]):
        for c in range(x.shape[1]):
            ref[y, c] = np.sort(xp[y:y + k, c:c + k].ravel())[(k * k - 1) // 2]
    assert np.array_equal(orc.medfilt(x, k), ref)


def test_median_rejects_bad_k(orc):
    with pytest.raises(ValueError):
        orc.medfilt(np.zeros((4, 4), np.float32), 4)


def test_r4_chained_median_replicates_stored_plane(orc):
    """R4: med7(med3(x)) uses the stored med3 plane's edges (library composition), which differs
    from evaluating med3 at virtual out-of-frame coordinates."""
    x = _rng(17).standard_normal((20, 20)).astype(np.float32)
    m3 = orc.medfilt(x, 3)
    ref = ndi.median_filter(ndi.median_filter(x, 3, mode="nearest"), 7, mode="nearest")
    assert np.array_equal(orc.medfilt(m3, 7), ref)


# ---------------------------------------------------------------- P4: dilation
@pytest.mark.parametrize("shape", [(1, 1), (1, 40), (33, 1), (40, 70)])
@pytest.mark.parametrize("density", [0.0, 0.02, 0.5, 1.0])
def test_p4_dilation_equals_scipy(orc, shape, density):
    m = (_rng(5).random(shape) < density).astype(np.uint8)
    ref = ndi.binary_dilation(m.astype(bool), structure=np.ones((3, 3), bool)).astype(np.uint8)
    assert np.array_equal(orc.dilate3(m), ref)


def test_p4_growth_gating_order(orc):
    """O6/R10 on the whole path: M2 = dil(M1) & G1, M3 = dil(M2) & G2, checked with scipy."""
    f = synth.make_frame(96, 96, seed=11, n_star=4, n_cr=40, n_hot=10)
    r = orc.run(f.img, debug_iter=0, **PARAMS)
    st = np.ones((3, 3), bool)
    m2 = ndi.binary_dilation(r["M1"].astype(bool), structure=st) & r["G1"].astype(bool)
    m3 = ndi.binary_dilation(m2, structure=st) & r["G2"].astype(bool)
    assert np.array_equal(r["M2"].astype(bool), m2)
    assert np.array_equal(r["M3"].astype(bool), m3)
    assert np.array_equal(r["C"].astype(bool), m3)           # first iteration: C = M3
    assert r["counts"][0] == m3.sum()


# ---------------------------------------------------------------- O2-O5: elementwise steps vs float64 closed forms
def test_elementwise_steps_against_float64_formulas(orc):
    f = synth.make_frame(80, 90, seed=12, n_star=5, n_cr=30, n_hot=10)
    p = dict(PARAMS, gain=1.7, readnoise=6.5)
    r = orc.run(f.img, debug_iter=0, **p)
    img = f.img.astype(np.float64)
    m5 = ndi.median_filter(f.img, 5, mode="nearest").astype(np.float64)
    N = np.sqrt(np.float32(1.7).astype(np.float64) * np.maximum(m5, 1e-4) +
                np.float64(np.float32(6.5)) ** 2) / np.float64(np.float32(1.7))
    assert np.allclose(r["N"], N, rtol=1e-6, atol=0)
    S = r["Lp"].astype(np.float64) / (2.0 * r["N"].astype(np.float64))
    assert np.allclose(r["S"], S, rtol=1e-6, atol=0)
    mS = ndi.median_filter(r["S"], 5, mode="nearest")
    assert np.array_equal(r["Sp"], r["S"] - mS)
    m3 = ndi.median_filter(f.img, 3, mode="nearest")
    m7 = ndi.median_filter(m3, 7, mode="nearest")
    assert np.array_equal(r["m3"], m3)
    assert np.array_equal(r["F"], np.maximum(m3 - m7, np.float32(0.01)))
    ok = f.img < np.float32(p["satlevel"])
    siglow = np.float32(p["sigfrac"]) * np.float32(p["sigclip"])
    assert np.array_equal(r["G1"].astype(bool), ok & (r["Sp"] > np.float32(p["sigclip"])))
    assert np.array_equal(r["G2"].astype(bool), ok & (r["Sp"] > siglow))
    ratio = r["Lp"] / r["F"]
    assert np.array_equal(r["M1"].astype(bool), r["G1"].astype(bool) & (ratio > np.float32(5.0)))
    assert img.shape == r["mask"].shape


# ---------------------------------------------------------------- P5: broad stars are never flagged
@pytest.mark.parametrize("fwhm", [2.5, 3.0, 4.0])
def test_p5_noise_free_broad_star_never_flagged(orc, fwhm):
    h = w = 41
    sg = fwhm / 2.35482
    for peak in (50.0, 500.0, 5000.0, 60000.0):
        for cy, cx in ((20.5, 20.5), (20.0, 20.0), (20.25, 20.7), (20.5, 20.0)):
            yy = (np.arange(h) + 0.5 - cy)[:, None]
            xx = (np.arange(w) + 0.5 - cx)[None, :]
            img = (100.0 + peak * np.exp(-(yy ** 2 + xx ** 2) / (2 * sg * sg))).astype(np.float32)
            r = orc.run(img, **PARAMS)
            assert not r["mask"].any(), (fwhm, peak, cy, cx)


def test_p5_sharp_source_is_flagged(orc):
    """Counter-check: an undersampled source (FWHM 1.0) IS flagged -- the test above can fail."""
    h = w = 41
    sg = 1.0 / 2.35482
    yy = (np.arange(h) + 0.5 - 20.5)[:, None]
    xx = (np.arange(w) + 0.5 - 20.5)[None, :]
    img = (100.0 + 5000.0 * np.exp(-(yy ** 2 + xx ** 2) / (2 * sg * sg))).astype(np.float32)
    assert orc.run(img, **PARAMS)["mask"].any()


# ---------------------------------------------------------------- P6: symmetry
def test_p6_rot180_and_flip_invariance(orc):
    f = synth.make_frame(120, 150, seed=21, n_star=10, n_cr=60, n_hot=20, sp_frac=0.003)
    r0 = orc.run(f.img, **PARAMS)
    for op in (lambda a: a[::-1, ::-1], lambda a: a[::-1, :], lambda a: a[:, ::-1]):
        r1 = orc.run(np.ascontiguousarray(op(f.img)), **PARAMS)
        assert np.array_equal(r1["mask"], op(r0["mask"]))
        assert np.array_equal(r1["clean"], op(r0["clean"]))
        assert np.array_equal(r1["counts"], r0["counts"])


# ---------------------------------------------------------------- P7: replacement is a pure function of (img, C)
def test_p7_clean_is_masked_median_of_input_and_final_mask(orc):
    f = synth.make_frame(128, 128, seed=31, n_star=8, n_cr=80, n_hot=20)
    r = orc.run(f.img, **PARAMS)
    keep = r["mask"] == 0
    assert np.array_equal(r["clean"][keep], f.img[keep])
    assert np.array_equal(r["clean"], orc.masked_median(f.img, r["mask"]))


# ---------------------------------------------------------------- P8: monotone mask, fixed point
def test_p8_monotone_and_fixed_point(orc):
    f = synth.make_frame(128, 128, seed=32, n_star=8, n_cr=80, n_hot=20)
    prev = None
    counts12 = orc.run(f.img, **dict(PARAMS, niter=12))["counts"]
    assert (counts12 == 0).any(), "iteration must reach a fixed point on this frame"
    t0 = int(np.argmax(counts12 == 0))
    assert (counts12[t0:] == 0).all()
    for n in range(0, t0 + 2):
        r = orc.run(f.img, **dict(PARAMS, niter=n))
        if prev is not None:
            assert not (prev & ~r["mask"].astype(bool)).any()      # C only grows
            assert r["mask"].sum() - prev.sum() == counts12[n - 1]
        prev = r["mask"].astype(bool)
    r_fix = orc.run(f.img, **dict(PARAMS, niter=t0 + 1))
    r_12 = orc.run(f.img, **dict(PARAMS, niter=12))
    assert np.array_equal(r_fix["mask"], r_12["mask"])
    assert np.array_equal(r_fix["clean"], r_12["clean"])


def test_niter_zero(orc):
    f = synth.make_frame(32, 32, seed=33, n_cr=10)
    r = orc.run(f.img, **dict(PARAMS, niter=0))
    assert not r["mask"].any() and np.array_equal(r["clean"], f.img)


# ---------------------------------------------------------------- P9: hand-computed replacement cases
def _golden_cases():
    cases, cur = [], None
    with open(os.path.join(GOLDEN, "masked_median_cases.txt")) as fh:
        for line in fh:
            t = line.split("#")[0].split()
            if not t:
                continue
            if t[0] == "case":
                cur = dict(name=t[1], mask=np.zeros((7, 7), np.uint8), expect=[])
                cases.append(cur)
            elif t[0] == "mask":
                for yx in t[1:]:
                    y, x = map(int, yx.split(","))
                    cur["mask"][y, x] = 1
            elif t[0] == "maskbox":
                y0, y1, x0, x1 = map(int, t[1:])
                cur["mask"][y0:y1 + 1, x0:x1 + 1] = 1
            elif t[0] == "expect":
                cur["expect"].append((int(t[1]), int(t[2]), float(t[3])))
    return cases


@pytest.mark.parametrize("case", _golden_cases(), ids=lambda c: c["name"])
def test_p9_hand_computed_masked_median(orc, case):
    img = (10 * np.arange(7)[:, None] + np.arange(7)[None, :]).astype(np.float32)
    out = orc.masked_median(img, case["mask"])
    assert len(case["expect"]) > 0
    for y, x, v in case["expect"]:
        assert out[y, x] == np.float32(v), (case["name"], y, x)
    keep = case["mask"] == 0
    assert np.array_equal(out[keep], img[keep])


def test_p9_masked_median_brute_force(orc):
    """Independent brute force with numpy on random masks (odd/even/zero donor counts, borders)."""
    rng = _rng(41)
    img = rng.standard_normal((14, 15)).astype(np.float32)
    mask = (rng.random(img.shape) < 0.45).astype(np.uint8)
    mask[0:6, 0:6] = 1                                       # a block with zero-donor pixels
    out = orc.masked_median(img, mask)
    ip, mp = np.pad(img, 2, mode="edge"), np.pad(mask, 2, mode="edge")
    n_zero = 0
    for y in range(img.shape[0]):
        for x in range(img.shape[1]):
            if not mask[y, x]:
                assert out[y, x] == img[y, x]
                continue
            v, m = ip[y:y + 5, x:x + 5].ravel(), mp[y:y + 5, x:x + 5].ravel()
            d = np.sort(v[m == 0])
            if d.size == 0:
                d = np.sort(v)
                n_zero += 1
            k = d.size
            ref = d[k // 2] if k % 2 else (d[k // 2 - 1] + d[k // 2]) * np.float32(0.5)
            assert out[y, x] == ref
    assert n_zero > 0


# ---------------------------------------------------------------- P10: saturation
def test_p10_saturated_plateau_never_masked(orc):
    f = synth.make_frame(200, 200, seed=51, n_star=10, n_cr=100, n_sat=12, sp_frac=0.01)
    assert f.sat_truth.sum() > 20
    r = orc.run(f.img, **PARAMS)
    assert not (r["mask"].astype(bool) & (f.img >= np.float32(65535.0))).any()
    # spike sitting at satlevel is never a candidate (R12) but is one with satlevel = +inf
    img = np.full((15, 15), 100.0, np.float32)
    img[7, 7] = 65535.0
    assert not orc.run(img, **PARAMS)["mask"].any()
    assert orc.run(img, **dict(PARAMS, satlevel=float("inf")))["mask"][7, 7] == 1


# ---------------------------------------------------------------- P11: negative image, zero read noise
def test_p11_negative_image_rn0_is_finite(orc):
    img = (-50.0 - 10.0 * _rng(61).random((30, 30))).astype(np.float32)
    r = orc.run(img, debug_iter=0, **dict(PARAMS, readnoise=0.0, gain=2.0))
    n = math.sqrt(2.0 * 1e-4) / 2.0
    assert np.allclose(r["N"], n, rtol=1e-6, atol=0)
    for k in ("Lp", "N", "S", "Sp", "F", "clean"):
        assert np.isfinite(r[k]).all(), k


# ---------------------------------------------------------------- P12: generator sanity (not parity)
def test_p12_generator_recall_and_determinism(orc):
    f = synth.make_config(0)
    g = synth.make_config(0)
    assert np.array_equal(f.img, g.img) and f.img.dtype == np.float32
    r = orc.run(f.img, **PARAMS)
    truth = f.cr_truth | f.hot_truth
    assert truth.sum() > 300
    assert r["mask"][truth].mean() > 0.97
    assert r["mask"].mean() < 0.02


def test_bad_arguments_rejected(orc):
    img = np.zeros((8, 8), np.float32)
    for bad in (dict(gain=-1.0), dict(gain=float("nan")), dict(readnoise=-1.0), dict(sigclip=0.0),
                dict(sigfrac=0.0), dict(objlim=-1.0), dict(niter=-1)):
        with pytest.raises(ValueError):
            orc.run(img, **dict(PARAMS, **bad))


# ------------------------------------------------------------------------------------------------
# R21: gain estimation when no gain is supplied (gain = 0).
def _sigma_clip_cases():
    cases, cur = [], None
    for ln in open(os.path.join(GOLDEN, "sigma_clip_cases.txt")):
        ln = ln.strip()
        if not ln or ln.startswith("#"):
            continue
        key, _, rest = ln.partition(" ")
        if key == "case":
            cur = dict(name=rest)
            cases.append(cur)
        elif key == "r":
            cur["r"] = [float(v) for v in rest.split()]
        elif key == "rounds":
            cur["rounds"] = int(rest)
        elif key == "expect":
            cur["expect"] = [float(v) for v in rest.split()]
    return cases


@pytest.mark.parametrize("case", _sigma_clip_cases(), ids=lambda c: c["name"])
def test_p13_hand_computed_sigma_clip(orc, case):
    s, stats = orc.sigma_clip(np.array(case["r"], np.float32), case["rounds"])
    c_e, s_e, lo_e, hi_e, kept_e = case["expect"]
    assert stats[0] == np.float32(c_e) and stats[4] == kept_e
    assert abs(s - s_e) <= 1e-6 * max(1.0, abs(s_e)) and abs(stats[1] - s_e) <= 1e-6 * max(1.0, abs(s_e))
    for got, exp in ((stats[2], lo_e), (stats[3], hi_e)):
        assert (got == exp) if math.isinf(exp) else abs(got - exp) <= 1e-5 * max(1.0, abs(exp))


def test_p13_sigma_clip_is_order_independent_and_rank_based(orc):
    """Selection only: any permutation of the input gives the same bits; the centre and the MAD are elements
    of fixed rank (library cross-check with np.partition on the first round)."""
    rng = np.random.default_rng(11)
    r = np.concatenate([rng.standard_normal(4001), 50 + 10 * rng.standard_normal(37)]).astype(np.float32)
    s0, st0 = orc.sigma_clip(r, 3)
    for _ in range(3):
        s1, st1 = orc.sigma_clip(rng.permutation(r), 3)
        assert s1 == s0 and np.array_equal(st1, st0)
    _, st = orc.sigma_clip(r, 1)
    k = (r.size - 1) // 2
    c = np.partition(r, k)[k]
    d = np.partition(np.abs(r - c), k)[k]
    assert st[0] == c and st[1] == np.float32(1.4826) * d
    assert 0.9 < s0 < 1.1 and st0[4] <= 4001 + 1          # the 50-sigma cluster is clipped away, sigma ~ 1


def _gain_cases():
    cases, cur = [], None
    for ln in open(os.path.join(GOLDEN, "gain_estimate_cases.txt")):
        ln = ln.strip()
        if not ln or ln.startswith("#"):
            continue
        key, _, rest = ln.partition(" ")
        if key == "case":
            cur = dict(name=rest, rows=[])
            cases.append(cur)
        elif key == "shape":
            cur["shape"] = tuple(int(v) for v in rest.split())
        elif key == "row":
            cur["rows"].append([float(v) for v in rest.split()])
        elif key == "rn":
            cur["rn"] = float(rest)
        elif key == "expect":
            cur["expect"] = [float(v) for v in rest.split()]
    return cases


@pytest.mark.parametrize("case", _gain_cases(), ids=lambda c: c["name"])
def test_p13_hand_computed_gain_estimate(orc, case):
    """tests/golden/gain_estimate_cases.txt: a frame small enough to do on paper, rn > 0, one clipped outlier whose
    med5 differs from the kept majority's.  Pins the read-noise root of R21 (the factor 4, the 2 s^2) and the
    restriction of the typical signal mt to the set the last clipping round kept."""
    img = np.array(case["rows"], np.float32)
    assert img.shape == case["shape"]
    g, st = orc.estimate_gain(img, case["rn"])
    g_e, c_e, s_e, lo_e, hi_e, kept_e, mt_e = case["expect"]
    assert st[0] == np.float32(c_e) and st[4] == kept_e and st[5] == np.float32(mt_e)
    assert abs(st[1] - s_e) <= 1e-6 * s_e
    assert abs(st[2] - lo_e) <= 1e-6 * abs(lo_e) and abs(st[3] - hi_e) <= 1e-6 * abs(hi_e)
    assert abs(float(g) - g_e) <= 2e-6 * g_e, (float(g), g_e)


@pytest.mark.parametrize("gain", [0.5, 2.0, 7.0])
def test_p13_gain_of_pure_poisson_like_noise_is_recovered(orc, gain):
    """Closed form behind R21: var(work) = signal/gain => (work - med5)/sqrt(med5) has sigma 1/sqrt(gain).  The
    pixel is part of its own median window, which lowers the residual variance by a few per cent."""
    rng = np.random.default_rng(5)
    B = 900.0
    img = (B + np.sqrt(B / gain) * rng.standard_normal((500, 620))).astype(np.float32)
    g, stats = orc.estimate_gain(img)
    assert abs(g / gain - 1.0) < 0.12
    assert abs(stats[0]) < 0.05 / math.sqrt(gain)
    assert g == np.float32(1.0) / (stats[1] * stats[1])          # no read noise: gain = 1/s^2 exactly
    assert abs(stats[5] / B - 1.0) < 0.01                         # typical signal = the sky level
    # robust: 1 % of the pixels hit by cosmic rays barely moves the estimate
    hit = rng.random(img.shape) < 0.01
    g2, _ = orc.estimate_gain(np.where(hit, img + 5000.0, img).astype(np.float32))
    assert abs(g2 / g - 1.0) < 0.05


@pytest.mark.parametrize("gain,rn,B", [(1.0, 10.0, 100.0), (2.0, 5.0, 400.0), (1.7, 20.0, 50.0), (0.6, 3.0, 30.0)])
def test_p13_gain_is_recovered_with_read_noise(orc, gain, rn, B):
    """The estimate must reproduce the noise model it feeds (O2): var(work) = B/gain + (rn/gain)^2.  Ignoring the
    read-noise term would read gain 0.54 for a true 1.0 at rn = 10 e- on a 100 ADU sky."""
    rng = np.random.default_rng(8)
    img = (B + np.sqrt(B / gain + (rn / gain) ** 2) * rng.standard_normal((500, 620))).astype(np.float32)
    g, _ = orc.estimate_gain(img, rn)
    assert abs(g / gain - 1.0) < 0.12
    g0, _ = orc.estimate_gain(img, 0.0)
    assert g0 < g                                                  # the read-noise term only raises the estimate


def test_p13_gain_scaling_is_exact(orc):
    """img -> 4 img scales every residual by exactly 2 (all operations scale by powers of two), hence
    gain -> gain / 4 bit for bit: pins the structure (difference over sqrt(median)) of the estimator."""
    f = synth.make_frame(96, 130, seed=4, n_star=5, n_cr=30, sp_frac=0.003)
    for rn in (0.0, 10.0):       # read noise is in electrons: unchanged when the image is rescaled
        g1, st1 = orc.estimate_gain(f.img, rn)
        g4, st4 = orc.estimate_gain(4.0 * f.img, rn)
        assert g4 * np.float32(4.0) == g1
        assert st4[0] == 2 * st1[0] and st4[1] == 2 * st1[1] and st4[4] == st1[4] and st4[5] == 4 * st1[5]


def test_p13_degenerate_and_whole_path(orc):
    g, stats = orc.estimate_gain(np.full((20, 30), 50.0, np.float32))
    assert g == 1.0 and stats[1] == 0.0                                     # sigma = 0 -> gain 1 (R21)
    f = synth.make_config(0)
    est = orc.run(f.img, **dict(PARAMS, gain=0.0))
    assert est["gains"].shape == (PARAMS["niter"],) and np.all(est["gains"] > 0)
    # iteration 0 estimates from the input frame; feeding the estimates back as supplied gains, one
    # iteration at a time, reproduces the run: the estimate only enters through the noise model
    g0, _ = orc.estimate_gain(f.img, PARAMS["readnoise"])
    assert est["gains"][0] == g0 and abs(g0 - 1.0) < 0.1                     # configs[0] was made with gain 1
    one = orc.run(f.img, **dict(PARAMS, gain=float(g0), niter=1))
    est1 = orc.run(f.img, **dict(PARAMS, gain=0.0, niter=1))
    assert np.array_equal(one["mask"], est1["mask"]) and np.array_equal(one["clean"], est1["clean"])
    g1, _ = orc.estimate_gain(est1["clean"], PARAMS["readnoise"])
    assert est["gains"][1] == g1                                            # iteration 1 sees the cleaned frame
    fixed = orc.run(f.img, **PARAMS)
    assert np.all(fixed["gains"] == np.float32(PARAMS["gain"]))
