"""Pins of the oracle's variant functions (readings R22-R26) against what the
mathematics fixes: library equivalents (scipy), brute force, closed forms, hand-worked golden cases and float64
re-evaluation of the defining formulas from the dumped planes.  All -m "not gpu"."""
import os

import numpy as np
import pytest
import scipy.ndimage as ndi

from paper_2602_17938_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
PARAMS = dict(synth.DEFAULT_PARAMS)


def _rng(seed):
    return np.random.Generator(np.random.Philox(seed))


# ------------------------------------------------------------------ orc_run_ex with no variant == orc_run
@pytest.mark.parametrize("gain", [1.0, 0.0])
def test_no_variant_equals_the_north_star_path(orc, gain):
    f = synth.make_frame(120, 150, seed=61, n_star=8, n_cr=80, n_hot=20, sp_frac=0.004, n_sat=2)
    p = dict(PARAMS, gain=gain)
    a = orc.run(f.img, debug_iter=1, **p)
    b = orc.run(f.img, debug_iter=1, fsmode=0, satgrow=-1, sepmed=0, **p)
    c = orc.run(f.img, debug_iter=1, bpm=np.zeros(f.img.shape, np.uint8), **p)
    for k in a:
        assert np.array_equal(a[k], b[k]), k
        assert np.array_equal(a[k], c[k]), k


# ------------------------------------------------------------------ R26: separable median
@pytest.mark.parametrize("k", [3, 5, 7])
def test_sepmed_equals_two_1d_library_medians(orc, k):
    rng = _rng(70 + k)
    for x in (rng.standard_normal((23, 31)).astype(np.float32),
              rng.integers(0, 3, (17, 40)).astype(np.float32),            # heavy ties
              rng.standard_normal((1, 9)).astype(np.float32), rng.standard_normal((9, 1)).astype(np.float32),
              rng.standard_normal((2, 2)).astype(np.float32)):
        ref = ndi.median_filter(ndi.median_filter(x, size=(1, k), mode="nearest"), size=(k, 1), mode="nearest")
        assert np.array_equal(orc.sepmedfilt(x, k), ref)


def test_sepmed_hand_case_differs_from_true_median(orc):
    """5x5 zeros with a 2x2 block of 9 at rows 1-2, cols 1-2; centre (2,2).  True 3x3 median: 4 nines of 9 -> 0.
    Row pass: T[1][1] = med(0,9,9) = 9, T[1][2] = med(9,9,0) = 9, T[1][3] = med(9,0,0) = 0; row 2 the same; row 3 all 0.
    Column pass at (2,2): med(T[1][2], T[2][2], T[3][2]) = med(9, 9, 0) = 9.  The approximation turns a corner pixel
    of the block into 9 where the true median says 0."""
    x = np.zeros((5, 5), np.float32)
    x[1:3, 1:3] = 9.0
    assert orc.medfilt(x, 3)[2, 2] == 0.0
    assert orc.sepmedfilt(x, 3)[2, 2] == 9.0
    assert orc.sepmedfilt(x, 3)[1, 3] == 0.0 and orc.sepmedfilt(x, 3)[1, 1] == 9.0


# ------------------------------------------------------------------ R25: extended saturated-star mask
@pytest.mark.parametrize("grow", [0, 1, 3])
def test_satstar_mask_equals_library_definition(orc, grow):
    f = synth.make_frame(150, 180, seed=62, n_star=10, n_cr=100, sp_frac=0.005, n_sat=12)
    assert (f.img >= 65535.0).sum() > 50
    core = ndi.median_filter(f.img, size=5, mode="nearest") >= np.float32(65535.0)
    ref = core if grow == 0 else ndi.binary_dilation(core, structure=np.ones((3, 3), bool), iterations=grow)
    got = orc.satstar_mask(f.img, 65535.0, grow)
    assert np.array_equal(got.astype(bool), ref) and got.sum() > 0


def test_satstar_mask_hand_cases(orc):
    """A 5x5 saturated block: a pixel is a core iff >= 13 of its 25 taps are saturated.  Offsets from the block centre:
    (0,0) 25; (0,+-1) 20; (+-1,+-1) 16; (0,+-2) 15; (+-1,+-2) 3x4 = 12 < 13; (+-2,+-2) 9; (0,+-3) 10.  Core = the inner
    3x3 plus the four edge midpoints = 13 pixels.  An isolated saturated pixel (1 of 25) is no core.  On the frame corner
    clamped taps count with multiplicity: a single saturated corner pixel holds 9 of the 25 taps -> no core; a 2x2
    saturated corner block holds 16 -> (0,0) is a core."""
    x = np.full((15, 15), 100.0, np.float32)
    x[5:10, 5:10] = 65535.0
    x[12, 2] = 65535.0
    exp = np.zeros((15, 15), bool)
    exp[6:9, 6:9] = True
    exp[7, 5] = exp[7, 9] = exp[5, 7] = exp[9, 7] = True
    assert np.array_equal(orc.satstar_mask(x, 65535.0, 0).astype(bool), exp)
    g1 = np.zeros((15, 15), bool)                     # one 3x3 dilation: the inner 3x3 grows to the 5x5 block (25) and
    g1[5:10, 5:10] = True                             # each arm tip adds the three pixels beyond its side (4 x 3) = 37
    g1[6:9, 4] = g1[6:9, 10] = g1[4, 6:9] = g1[10, 6:9] = True
    assert np.array_equal(orc.satstar_mask(x, 65535.0, 1).astype(bool), g1) and g1.sum() == 37
    y = np.full((9, 9), 100.0, np.float32)
    y[0, 0] = 65535.0
    assert orc.satstar_mask(y, 65535.0, 0).sum() == 0
    y[0:2, 0:2] = 65535.0
    m = orc.satstar_mask(y, 65535.0, 0)
    assert m[0, 0] == 1 and m[2, 2] == 0
    assert orc.satstar_mask(y, float("inf"), 2).sum() == 0           # nothing reaches +inf


# ------------------------------------------------------------------ R23: bad pixels in the replacement
def _bpm_cases():
    cases, cur = [], None
    with open(os.path.join(GOLDEN, "masked_median_bpm_cases.txt")) as fh:
        for line in fh:
            t = line.split("#")[0].split()
            if not t:
                continue
            if t[0] == "case":
                cur = dict(name=t[1], mask=np.zeros((7, 7), np.uint8), bpm=np.zeros((7, 7), np.uint8), expect=[])
                cases.append(cur)
            elif t[0] in ("mask", "bpm"):
                for yx in t[1:]:
                    y, x = map(int, yx.split(","))
                    cur[t[0]][y, x] = 1
            elif t[0] in ("maskbox", "bpmbox"):
                y0, y1, x0, x1 = map(int, t[1:])
                cur[t[0][:-3]][y0:y1 + 1, x0:x1 + 1] = 1
            elif t[0] == "expect":
                cur["expect"].append((int(t[1]), int(t[2]), float(t[3])))
    return cases


@pytest.mark.parametrize("case", _bpm_cases(), ids=lambda c: c["name"])
def test_hand_computed_masked_median_with_bad_pixels(orc, case):
    img = (10 * np.arange(7)[:, None] + np.arange(7)[None, :]).astype(np.float32)
    out = orc.masked_median_bpm(img, case["mask"], case["bpm"])
    assert len(case["expect"]) > 0
    for y, x, v in case["expect"]:
        assert out[y, x] == np.float32(v), (case["name"], y, x, out[y, x])
    keep = case["mask"] == 0
    assert np.array_equal(out[keep], img[keep])


def test_masked_median_with_bad_pixels_brute_force(orc):
    rng = _rng(43)
    img = rng.standard_normal((16, 13)).astype(np.float32)
    mask = (rng.random(img.shape) < 0.3).astype(np.uint8)
    bpm = ((rng.random(img.shape) < 0.3) & (mask == 0)).astype(np.uint8)
    mask[0:5, 0:5] = 1
    bpm[0:7, 0:7] |= (mask[0:7, 0:7] == 0)                       # zero-donor pixels around the corner
    out = orc.masked_median_bpm(img, mask, bpm)
    ip, mp, bp = (np.pad(a, 2, mode="edge") for a in (img, mask, bpm))
    nzero = 0
    for y in range(img.shape[0]):
        for x in range(img.shape[1]):
            if not mask[y, x]:
                assert out[y, x] == img[y, x]
                continue
            wv, wm, wb = ip[y:y + 5, x:x + 5].ravel(), mp[y:y + 5, x:x + 5].ravel(), bp[y:y + 5, x:x + 5].ravel()
            don = np.sort(wv[(wm == 0) & (wb == 0)])
            if don.size == 0:
                don = np.sort(wv)
                nzero += 1
            k = don.size
            exp = don[k // 2] if k & 1 else np.float32((don[k // 2 - 1] + don[k // 2]) * np.float32(0.5))
            assert out[y, x] == exp, (y, x)
    assert nzero > 0
    assert np.array_equal(orc.masked_median_bpm(img, mask, None), orc.masked_median(img, mask))


def test_bad_pixels_on_the_whole_path(orc):
    """R23: a bad pixel is never flagged (even a 5000-ADU spike), never a donor; everything else follows.  P7 with the
    bad pixels: clean == masked_median_bpm(img, final mask, bpm)."""
    f = synth.make_frame(140, 170, seed=63, n_star=8, n_cr=120, n_hot=30, sp_frac=0.004)
    base = orc.run(f.img, **PARAMS)
    ys, xs = np.nonzero(base["mask"])
    bpm = np.zeros(f.img.shape, np.uint8)
    bpm[ys[::3], xs[::3]] = 1                                      # a third of the flagged pixels declared bad
    bpm[_rng(5).random(f.img.shape) < 0.01] = 1
    r = orc.run(f.img, bpm=bpm, **PARAMS)
    assert not (r["mask"] & bpm).any() and r["mask"].sum() > 0
    assert np.array_equal(r["clean"][bpm != 0], f.img[bpm != 0])
    assert np.array_equal(r["clean"], orc.masked_median_bpm(f.img, r["mask"], bpm))
    assert not np.array_equal(r["clean"], orc.masked_median(f.img, r["mask"]))      # the donor rule matters here
    assert int(r["counts"].sum()) == int(r["mask"].sum())


# ------------------------------------------------------------------ R24: variance plane
def test_variance_plane_closed_forms(orc):
    """Constant variance v: N = sqrt(v) everywhere, so an isolated spike of height A on a flat frame has S = S' = A/sqrt(v)
    (L+ = 2A, P2) and is flagged iff A/sqrt(v) > sigclip.  v <= 1e-8 is floored: N = 1e-4."""
    B, v = 50.0, 25.0
    for A, flagged in ((4.4 * 5.0, False), (4.6 * 5.0, True)):
        img = np.full((21, 23), B, np.float32)
        img[10, 11] += A
        r = orc.run(img, debug_iter=0, var=np.full(img.shape, v, np.float32), **PARAMS)
        assert np.all(r["N"] == np.float32(5.0))
        assert r["S"][10, 11] == np.float32(2 * A) / np.float32(10.0) and r["Sp"][10, 11] == r["S"][10, 11]
        assert bool(r["mask"][10, 11]) == flagged and r["mask"].sum() == int(flagged)
    img = np.full((9, 9), B, np.float32)
    r = orc.run(img, debug_iter=0, var=np.zeros(img.shape, np.float32), **PARAMS)
    assert np.all(r["N"] == np.float32(1e-4)) and r["mask"].sum() == 0
    r = orc.run(img, debug_iter=0, var=np.full(img.shape, -3.0, np.float32), **PARAMS)
    assert np.all(r["N"] == np.float32(1e-4))


def test_variance_plane_equal_to_the_noise_model_reproduces_it(orc):
    """Spikes on a flat sky B = 96 with gain 1, rn = 10: med5 = B everywhere in every iteration, so the model's N is
    sqrt(96 + 100) = 14 exactly; the variance plane 196 gives the same N and therefore identical outputs."""
    rng = _rng(64)
    img = np.full((80, 90), 96.0, np.float32)
    ys, xs = rng.integers(3, 77, 40), rng.integers(3, 87, 40)
    keep = [i for i in range(40) if all(max(abs(ys[i] - ys[j]), abs(xs[i] - xs[j])) > 6 for j in range(i))]
    img[ys[keep], xs[keep]] += rng.uniform(30, 3000, len(keep)).astype(np.float32)
    a = orc.run(img, debug_iter=0, **PARAMS)
    b = orc.run(img, debug_iter=0, var=np.full(img.shape, 196.0, np.float32), **dict(PARAMS, gain=0.0))
    assert np.all(a["N"] == np.float32(14.0)) and a["mask"].sum() > 10
    for k in ("N", "S", "Sp", "F", "G1", "G2", "M1", "M3", "mask", "clean", "counts"):
        assert np.array_equal(a[k], b[k]), k


# ------------------------------------------------------------------ R22: noise-normalised fine structure
def test_normalised_fine_structure_against_float64_formulas(orc):
    """Fn = max((m3 - m7)/N, 0.01) and M1 = G1 and (S'/Fn > objlim), re-evaluated in float64 from the dumped planes
    (values within 1e-5 relative of a threshold excluded from the exact comparison, and counted)."""
    f = synth.make_frame(160, 200, seed=65, n_star=14, n_cr=150, n_hot=30, sp_frac=0.004)
    for it in (0, 1):
        r = orc.run(f.img, debug_iter=it, fsmode=1, **PARAMS)
        m3 = ndi.median_filter(r["work_in"], size=3, mode="nearest")
        m7 = ndi.median_filter(m3, size=7, mode="nearest")
        assert np.array_equal(r["m3"], m3)
        fn = np.maximum((m3.astype(np.float64) - m7) / r["N"].astype(np.float64), 0.01)
        assert np.allclose(r["F"], fn, rtol=3e-7, atol=0)
        ratio = r["Sp"].astype(np.float64) / r["F"].astype(np.float64)
        sure = np.abs(ratio - PARAMS["objlim"]) > 1e-5 * PARAMS["objlim"]
        exp = (r["G1"] != 0) & (ratio > PARAMS["objlim"])
        assert np.array_equal((r["M1"] != 0)[sure], exp[sure]) and (~sure & (r["G1"] != 0)).sum() < 3
        assert r["M1"].sum() > 50 and (r["G1"] & ~r["M1"] & 1).sum() > 0          # both outcomes occur


def test_normalised_fine_structure_halves_the_contrast(orc):
    """Where med5(S) = 0 and F is above its floor, S'/Fn = (L+/(2N)) / (F/N) = (L+/F)/2: the noise-normalised test is the
    north-star test with twice the objlim (up to rounding).  Frame: flat sky, isolated 5x5 plateaus of height f = 40 with a
    spike of height A on the centre: there L+ = 2A, m3 = B + f, m7 = B, F = f = 40 ADU (worked out in DESIGN.md R22)."""
    B, fobj = 100.0, 40.0
    img = np.full((40, 120), B, np.float32)
    amps = [100.0, 150.0, 250.0, 400.0, 1000.0]                   # L+/F = 2A/f = 5, 7.5, 12.5, 20, 50
    for i, A in enumerate(amps):
        x0 = 10 + 22 * i
        img[18:23, x0:x0 + 5] += fobj
        img[20, x0 + 2] += A
    a = orc.run(img, debug_iter=0, fsmode=0, **PARAMS)
    b = orc.run(img, debug_iter=0, fsmode=1, **PARAMS)
    for i, A in enumerate(amps):
        y, x = 20, 10 + 22 * i + 2
        assert a["Lp"][y, x] == np.float32(2 * A) and a["F"][y, x] == np.float32(fobj)
        r0 = a["Lp"][y, x] / a["F"][y, x]
        r1 = b["Sp"][y, x] / b["F"][y, x]
        mS = b["S"][y, x] - b["Sp"][y, x]
        # med5(S) at the centre is the small S of the plateau's edge pixels; correct for it exactly
        assert abs((r1 + mS / b["F"][y, x]) / (r0 / 2) - 1.0) < 1e-6
        assert bool(a["M1"][y, x]) == (r0 > 5.0) and bool(b["M1"][y, x]) == (r1 > 5.0)
    # decisions: objlim = 5 -> R7 flags 2A/f > 5 (all but the first), R22 flags roughly A/f > 5 (the last three at most)
    got0 = [bool(a["M1"][20, 10 + 22 * i + 2]) for i in range(5)]
    got1 = [bool(b["M1"][20, 10 + 22 * i + 2]) for i in range(5)]
    assert got0 == [False, True, True, True, True]
    assert got1 == [False, False, True, True, True]


# ------------------------------------------------------------------ R25 on the whole path
def test_satstar_mask_on_the_whole_path(orc):
    f = synth.make_frame(200, 240, seed=66, n_star=10, n_cr=150, sp_frac=0.01, n_sat=16)
    p = dict(PARAMS, satlevel=60000.0)
    base = orc.run(f.img, **p)
    for grow in (0, 2):
        nok = orc.satstar_mask(f.img, 60000.0, grow)
        r = orc.run(f.img, satgrow=grow, **p)
        assert nok.sum() > 30 and not (r["mask"] & nok).any()
        # outside the reach of the protected pixels (growth 2 px, replacement windows 2 px per iteration) nothing changes
        far = ~ndi.binary_dilation(nok.astype(bool), structure=np.ones((3, 3), bool), iterations=4 * 8 + 6)
        assert np.array_equal(r["mask"][far], base["mask"][far])
    assert (orc.run(f.img, satgrow=4, **p)["mask"] & orc.satstar_mask(f.img, 60000.0, 4)).sum() == 0


# ------------------------------------------------------------------ R26 on the whole path
def test_sepmed_whole_path_planes(orc):
    """Every median of O2-O4 is the separable one: re-derive the dumped planes with the library's 1-D medians."""
    f = synth.make_frame(130, 160, seed=67, n_star=10, n_cr=100, sp_frac=0.005, n_sat=3)

    def sep(x, k):
        return ndi.median_filter(ndi.median_filter(x, size=(1, k), mode="nearest"), size=(k, 1), mode="nearest")
    r = orc.run(f.img, debug_iter=1, sepmed=1, **PARAMS)
    w = r["work_in"]
    m5 = np.maximum(sep(w, 5), np.float32(1e-4))
    assert np.array_equal(r["N"], np.sqrt(m5 + np.float32(100.0), dtype=np.float32))     # gain 1: N = sqrt(m5 + rn^2)
    assert np.array_equal(r["m3"], sep(w, 3))
    assert np.array_equal(r["F"], np.maximum(r["m3"] - sep(r["m3"], 7), np.float32(0.01)))
    assert np.array_equal(r["Sp"], r["S"] - sep(r["S"], 5))
    t = orc.run(f.img, **PARAMS)
    assert not np.array_equal(t["mask"], orc.run(f.img, sepmed=1, **PARAMS)["mask"])


def test_sepmed_flags_near_saturated_star_cores_the_true_median_does_not(orc):
    """PAPER.md:29 'the use of a separable median filter can result in the incorrect removal of cosmic rays by incorrectly
    classifying the center of near-saturated or saturated stars as cosmic rays' -- on a configs[4]-like frame (stress
    stars with peaks 40000-80000, plateaus clipped at 65535) the true median flags no pixel at or above 40000 ADU, the
    separable one does."""
    f = synth.make_frame(600, 800, seed=5, n_star=60, n_cr=300, sp_frac=0.01, n_sat=30)
    bright = f.img >= np.float32(40000.0)
    assert bright.sum() > 1000
    for sat in (65535.0, float("inf")):
        p = dict(PARAMS, satlevel=sat)
        t = orc.run(f.img, **p)["mask"].astype(bool)
        s = orc.run(f.img, sepmed=1, **p)["mask"].astype(bool)
        print("satlevel %s: star-core pixels (>= 40000 ADU) flagged: true median %d, separable median %d of %d"
              % (sat, (t & bright).sum(), (s & bright).sum(), bright.sum()))
        assert (t & bright).sum() == 0
        assert (s & bright).sum() > 0
