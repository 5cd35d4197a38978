"""ctypes loader for the CPU oracle (oracle/lacosmic_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2602_17938_b200 (the CUDA path) and the
CUDA path imports nothing from here.  Every function is argument marshalling around the C
routine of the same name; the arithmetic lives in the C file, which cites the passages it
follows (BASELINE.json north_star (1)-(7)).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lacosmic_oracle.c")
_LIB = os.path.join(_HERE, "liblacosmic_oracle.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-std=c99"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no -ffast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Debug(C.Structure):
    _fields_ = [("iter", C.c_int)] + \
        [(n, C.c_void_p) for n in ("Lp", "N", "S", "Sp", "m3", "F")] + \
        [(n, C.c_void_p) for n in ("G1", "G2", "M1", "M2", "M3", "C")] + \
        [("work_in", C.c_void_p)]


_F32_PLANES = ("Lp", "N", "S", "Sp", "m3", "F", "work_in")
_U8_PLANES = ("G1", "G2", "M1", "M2", "M3", "C")
_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        fp, u8p, i32p = C.c_void_p, C.c_void_p, C.c_void_p
        L.orc_lplus.argtypes = [fp, fp, C.c_int, C.c_int]
        L.orc_lplus.restype = None
        L.orc_medfilt.argtypes = [fp, fp, C.c_int, C.c_int, C.c_int]
        L.orc_medfilt.restype = C.c_int
        L.orc_dilate3.argtypes = [u8p, u8p, C.c_int, C.c_int]
        L.orc_dilate3.restype = None
        L.orc_masked_median.argtypes = [fp, u8p, fp, C.c_int, C.c_int]
        L.orc_masked_median.restype = None
        L.orc_run.argtypes = [fp, C.c_int, C.c_int] + [C.c_float] * 5 + [C.c_int, C.c_float,
                                                                        u8p, fp, i32p, C.c_void_p, fp]
        L.orc_estimate_gain.argtypes = [fp, C.c_int, C.c_int, C.c_float, fp, fp]
        L.orc_estimate_gain.restype = C.c_int
        L.orc_sigma_clip.argtypes = [fp, C.c_size_t, C.c_int, fp]
        L.orc_sigma_clip.restype = C.c_float
        L.orc_run.restype = C.c_int
        L.orc_sepmedfilt.argtypes = [fp, fp, C.c_int, C.c_int, C.c_int]
        L.orc_sepmedfilt.restype = C.c_int
        L.orc_satstar_mask.argtypes = [fp, C.c_int, C.c_int, C.c_float, C.c_int, u8p]
        L.orc_satstar_mask.restype = C.c_int
        L.orc_masked_median_bpm.argtypes = [fp, u8p, u8p, fp, C.c_int, C.c_int]
        L.orc_masked_median_bpm.restype = None
        L.orc_run_ex.argtypes = [fp, C.c_int, C.c_int] + [C.c_float] * 5 + [C.c_int, C.c_float, C.c_void_p,
                                                                           u8p, fp, i32p, C.c_void_p, fp]
        L.orc_run_ex.restype = C.c_int
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_get_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    assert a.ndim == 2
    return a


def _u8(a):
    a = np.ascontiguousarray(a).astype(np.uint8, copy=False)
    assert a.ndim == 2
    return np.ascontiguousarray(a)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def max_threads() -> int:
    return int(lib().orc_get_max_threads())


def lplus(img):
    img = _f32(img)
    out = np.empty_like(img)
    lib().orc_lplus(_p(img), _p(out), *img.shape)
    return out


def medfilt(img, k):
    img = _f32(img)
    out = np.empty_like(img)
    rc = lib().orc_medfilt(_p(img), _p(out), img.shape[0], img.shape[1], int(k))
    if rc != 0:
        raise ValueError("orc_medfilt: bad argument (k must be 3, 5 or 7)")
    return out


def dilate3(mask):
    mask = _u8(mask)
    out = np.empty_like(mask)
    lib().orc_dilate3(_p(mask), _p(out), *mask.shape)
    return out


def masked_median(img, mask):
    img, mask = _f32(img), _u8(mask)
    assert img.shape == mask.shape
    out = np.empty_like(img)
    lib().orc_masked_median(_p(img), _p(mask), _p(out), *img.shape)
    return out


def sepmedfilt(img, k):
    """R26: separable k x k median (row pass, then column pass); comparison only."""
    img = _f32(img)
    out = np.empty_like(img)
    rc = lib().orc_sepmedfilt(_p(img), _p(out), img.shape[0], img.shape[1], int(k))
    if rc != 0:
        raise ValueError("orc_sepmedfilt: bad argument")
    return out


def satstar_mask(img, satlevel=65535.0, grow=0):
    """R25: (med5(img) >= satlevel) dilated `grow` times by the 3x3 square."""
    img = _f32(img)
    out = np.empty(img.shape, np.uint8)
    rc = lib().orc_satstar_mask(_p(img), img.shape[0], img.shape[1], float(satlevel), int(grow), _p(out))
    if rc != 0:
        raise ValueError("orc_satstar_mask: bad argument")
    return out


def masked_median_bpm(img, mask, bpm=None):
    """O7 with bad pixels removed from the donors (R23)."""
    img, mask = _f32(img), _u8(mask)
    out = np.empty_like(img)
    b = None if bpm is None else _u8(bpm)
    lib().orc_masked_median_bpm(_p(img), _p(mask), None if b is None else _p(b), _p(out), *img.shape)
    return out


class _Variant(C.Structure):
    _fields_ = [("fsmode", C.c_int), ("satgrow", C.c_int), ("sepmed", C.c_int), ("bpm", C.c_void_p),
                ("var", C.c_void_p)]


def sigma_clip(r, rounds=3):
    """R21 sigma clipping of a 1-D fp32 vector.  Returns (s, stats = [c, s, lo, hi, kept] of the last round)."""
    r = np.ascontiguousarray(r, dtype=np.float32).ravel()
    stats = np.zeros(5, np.float32)
    s = lib().orc_sigma_clip(_p(r), r.size, int(rounds), _p(stats))
    return float(np.float32(s)), stats


def estimate_gain(img, readnoise=0.0):
    """R21 gain estimate of one image.  Returns (gain fp32, stats = [c, s, lo, hi, kept, mt])."""
    img = _f32(img)
    g = np.zeros(1, np.float32)
    stats = np.zeros(6, np.float32)
    rc = lib().orc_estimate_gain(_p(img), img.shape[0], img.shape[1], float(readnoise), _p(g), _p(stats))
    if rc != 0:
        raise ValueError("orc_estimate_gain failed with code %d" % rc)
    return np.float32(g[0]), stats


def run(img, gain=1.0, readnoise=10.0, sigclip=4.5, sigfrac=0.3, objlim=5.0, niter=4,
        satlevel=65535.0, debug_iter=None, fsmode=None, satgrow=None, sepmed=None, bpm=None, var=None):
    """Whole path (O0-O7).  gain = 0: estimated at each iteration (R21).  Returns dict(mask=u8, clean=f32,
    counts=int32[niter], gains=f32[niter] (the gain each iteration used), [debug planes]).
    Any of fsmode / satgrow / sepmed / bpm / var given: orc_run_ex with those variants (R22-R26); none given:
    orc_run, the north-star path."""
    img = _f32(img)
    h, w = img.shape
    mask = np.empty((h, w), np.uint8)
    clean = np.empty((h, w), np.float32)
    counts = np.zeros(max(niter, 1), np.int32)
    out = {}
    dbg_ref = None
    if debug_iter is not None:
        dbg = _Debug()
        dbg.iter = int(debug_iter)
        for n in _F32_PLANES:
            out[n] = np.zeros((h, w), np.float32)
            setattr(dbg, n, out[n].ctypes.data)
        for n in _U8_PLANES:
            out[n] = np.zeros((h, w), np.uint8)
            setattr(dbg, n, out[n].ctypes.data)
        dbg_ref = C.byref(dbg)
    gains = np.zeros(max(niter, 1), np.float32)
    if all(a is None for a in (fsmode, satgrow, sepmed, bpm, var)):
        rc = lib().orc_run(_p(img), h, w, gain, readnoise, sigclip, sigfrac, objlim, int(niter),
                           satlevel, _p(mask), _p(clean), _p(counts), dbg_ref, _p(gains))
    else:
        b = None if bpm is None else _u8(bpm)
        vp = None if var is None else _f32(var)
        assert (b is None or b.shape == img.shape) and (vp is None or vp.shape == img.shape)
        v = _Variant(int(fsmode or 0), -1 if satgrow is None else int(satgrow), int(bool(sepmed)),
                     None if b is None else b.ctypes.data, None if vp is None else vp.ctypes.data)
        rc = lib().orc_run_ex(_p(img), h, w, gain, readnoise, sigclip, sigfrac, objlim, int(niter),
                              satlevel, C.byref(v), _p(mask), _p(clean), _p(counts), dbg_ref, _p(gains))
    if rc != 0:
        raise ValueError("orc_run failed with code %d" % rc)
    out.update(mask=mask, clean=clean, counts=counts[:niter].copy(), gains=gains[:niter].copy())
    return out
