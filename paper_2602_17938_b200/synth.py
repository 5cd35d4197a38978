"""Seeded synthetic MOTHRA-shaped frames (input generator only).

This module holds NONE of the method's arithmetic: it only draws the inputs
that both the CUDA path and the CPU oracle consume (tier rule (3): "only the
seeded input generators serve both, from a module of their own").  It imports
numpy and nothing else from this repository.

Recipe G(h, w, seed, n_star, n_cr, n_hot, sp_frac, n_sat) follows SURVEY.md
section 8(d) / BASELINE.json `configs`; the frames stand in for the astroscrappy
mock data and the MOTHRA frames of PAPER.md:31,47, which are not available.
All draws come from ``numpy.random.Generator(numpy.random.Philox(seed))`` in the
fixed order written below, in float64; the frame is cast to fp32 last.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

SKY_ADU = 100.0
GAIN = 1.0
READNOISE = 10.0
SATLEVEL = 65535.0
FWHM_TO_SIGMA = 2.35482

# Parameters quoted by every BASELINE.json config.
DEFAULT_PARAMS = dict(gain=1.0, readnoise=10.0, sigclip=4.5, sigfrac=0.3,
                      objlim=5.0, niter=4, satlevel=65535.0)


@dataclass
class Frame:
    img: np.ndarray          # fp32 [h][w]
    cr_truth: np.ndarray     # bool [h][w]: injected cosmic-ray pixels
    hot_truth: np.ndarray    # bool [h][w]: injected hot pixels
    sp_truth: np.ndarray     # int8 [h][w]: +1 / -1 salt-and-pepper outliers
    sat_truth: np.ndarray    # bool [h][w]: pixels clipped at satlevel


def _stamp_gaussians(signal, ys, xs, sigmas, peaks):
    h, w = signal.shape
    for cy, cx, sg, pk in zip(ys, xs, sigmas, peaks):
        rad = int(math.ceil(6.0 * sg)) + 1
        y0 = max(int(math.floor(cy)) - rad, 0)
        y1 = min(int(math.floor(cy)) + rad + 1, h)
        x0 = max(int(math.floor(cx)) - rad, 0)
        x1 = min(int(math.floor(cx)) + rad + 1, w)
        if y1 <= y0 or x1 <= x0:
            continue
        # point-sampled at pixel centres (pixel (j,i) has centre (j+0.5, i+0.5))
        yy = (np.arange(y0, y1, dtype=np.float64) + 0.5 - cy)[:, None]
        xx = (np.arange(x0, x1, dtype=np.float64) + 0.5 - cx)[None, :]
        signal[y0:y1, x0:x1] += pk * np.exp(-(yy * yy + xx * xx) / (2.0 * sg * sg))


def make_frame(h, w, seed, n_star=0, n_cr=0, n_hot=0, sp_frac=0.0, n_sat=0) -> Frame:
    rng = np.random.Generator(np.random.Philox(int(seed)))
    # 1. sky
    signal = np.full((h, w), SKY_ADU, dtype=np.float64)
    # 2. stars
    sy = rng.uniform(0.0, h, n_star)
    sx = rng.uniform(0.0, w, n_star)
    fwhm = rng.uniform(2.5, 4.0, n_star)
    peak = np.exp(rng.uniform(math.log(50.0), math.log(30000.0), n_star))
    _stamp_gaussians(signal, sy, sx, fwhm / FWHM_TO_SIGMA, peak)
    # 3. (near-)saturated stress stars
    if n_sat:
        ty = rng.uniform(0.0, h, n_sat)
        tx = rng.uniform(0.0, w, n_sat)
        tpeak = rng.uniform(40000.0, 80000.0, n_sat)
        tw = rng.integers(3, 10, n_sat)                 # plateau width 3..9 px
        tfwhm = rng.uniform(2.5, 4.0, n_sat)
        tsig = tfwhm / FWHM_TO_SIGMA
        over = tpeak > SATLEVEL
        tsig[over] = np.minimum(
            (tw[over] / 2.0) / np.sqrt(2.0 * np.log(tpeak[over] / SATLEVEL)), 8.0)
        _stamp_gaussians(signal, ty, tx, tsig, tpeak)
    # 4. Gaussian stand-in for Poisson + read noise
    img = signal + rng.standard_normal((h, w)) * np.sqrt(
        np.maximum(signal, 0.0) / GAIN + (READNOISE / GAIN) ** 2)
    del signal
    # 5. cosmic rays: single pixels and straight tracks
    cr_truth = np.zeros((h, w), dtype=bool)
    cy = rng.integers(0, h, n_cr)
    cx = rng.integers(0, w, n_cr)
    amp = rng.uniform(500.0, 10000.0, n_cr)
    single = rng.random(n_cr) < 0.5
    length = rng.integers(2, 7, n_cr)
    theta = rng.uniform(0.0, math.pi, n_cr)
    for i in range(n_cr):
        n = 1 if single[i] else int(length[i])
        st, ct = math.sin(theta[i]), math.cos(theta[i])
        seen = set()
        for t in range(n):
            y = int(round(cy[i] + t * st))
            x = int(round(cx[i] + t * ct))
            if 0 <= y < h and 0 <= x < w and (y, x) not in seen:
                seen.add((y, x))
                img[y, x] += amp[i]
                cr_truth[y, x] = True
    # 6. isolated hot pixels (rejected if within Chebyshev distance 2 of a defect)
    hot_truth = np.zeros((h, w), dtype=bool)
    hy = rng.integers(0, h, n_hot)
    hx = rng.integers(0, w, n_hot)
    hamp = rng.uniform(200.0, 5000.0, n_hot)
    for i in range(n_hot):
        y, x = int(hy[i]), int(hx[i])
        y0, y1, x0, x1 = max(y - 2, 0), min(y + 3, h), max(x - 2, 0), min(x + 3, w)
        if cr_truth[y0:y1, x0:x1].any() or hot_truth[y0:y1, x0:x1].any():
            continue
        img[y, x] += hamp[i]
        hot_truth[y, x] = True
    # 7. CMOS salt-and-pepper
    sp_truth = np.zeros((h, w), dtype=np.int8)
    if sp_frac > 0.0:
        hit = rng.random((h, w)) < sp_frac
        k = int(hit.sum())
        sigma_sky = math.sqrt(SKY_ADU / GAIN + (READNOISE / GAIN) ** 2)
        mag = rng.uniform(5.0, 50.0, k) * sigma_sky
        sign = np.where(rng.random(k) < 0.5, -1.0, 1.0)
        img[hit] += sign * mag
        sp_truth[hit] = sign.astype(np.int8)
    # 8. clip at satlevel; fp32 last.  No lower clip: negative pixels are legal.
    sat_truth = img >= SATLEVEL
    np.minimum(img, SATLEVEL, out=img)
    return Frame(img.astype(np.float32), cr_truth, hot_truth, sp_truth, sat_truth)


# BASELINE.json configs[i] -> generator arguments.
CONFIGS = {
    0: dict(h=512, w=512, seed=1, n_star=100, n_cr=300, n_hot=100),
    1: dict(h=2048, w=2048, seed=2, n_star=1500, n_cr=5000, n_hot=2000),
    2: dict(h=4000, w=6500, seed=3, n_star=8000, n_cr=30000, sp_frac=0.005),
    4: dict(h=4000, w=6500, seed=5, n_star=8000, n_cr=30000, sp_frac=0.01, n_sat=300),
}


def make_config(i: int, **override) -> Frame:
    """Frame of BASELINE.json configs[i] (i in 0, 1, 2, 4)."""
    kw = dict(CONFIGS[i])
    kw.update(override)
    return make_frame(**kw)


def _image(kw):
    return make_frame(**kw).img


def make_images(kws, workers=None):
    """The fp32 images make_frame(**kw).img for kw in kws, in order, drawn in worker processes (bench.py's 64-frame
    stream: a 4000 x 6500 frame takes about 3 s of one core).  The workers are SPAWNED, not forked, so this is safe in a
    process that has already initialised CUDA; each draw is seeded by its own kw, so the result does not depend on the
    number of workers."""
    import multiprocessing as mp
    import os
    from concurrent.futures import ProcessPoolExecutor
    kws = list(kws)
    workers = min(len(kws), workers or min(16, os.cpu_count() or 1))
    if workers <= 1:
        for kw in kws:
            yield _image(kw)
        return
    with ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as ex:
        for img in ex.map(_image, kws):
            yield img


def stream_config(n_frames=64, h=4000, w=6500, first_seed=1000):
    """configs[3]: per-frame (seed, params) of the 64-frame stream.

    Frames come from the configs[2] generator with seeds 1000..1063; sigclip
    cycles over {4.0, 4.5, 5.0} by seed mod 3 ("per-frame parameters").
    """
    out = []
    for j in range(n_frames):
        seed = first_seed + j
        p = dict(DEFAULT_PARAMS)
        p["sigclip"] = (4.0, 4.5, 5.0)[seed % 3]
        kw = dict(CONFIGS[2])
        kw.update(h=h, w=w, seed=seed)
        out.append((kw, p))
    return out
