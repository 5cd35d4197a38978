"""ctypes binding of include/lacosmic.h -- same names, argument marshalling only.

Device buffers are torch CUDA tensors (torch = device memory + streams, nothing else); every step
of the path runs inside liblacosmic_b200.so.  The library must exist: a missing or unloadable
library raises LacosmicError (there is deliberately no fallback of any kind).
"""
from __future__ import annotations

import ctypes as C
import functools
import os
from dataclasses import dataclass

MAX_NITER = 64
_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "liblacosmic_b200.so")
_lib = None

EXPORTS = (
    "lacosmic_run", "lacosmic_workspace_bytes", "lacosmic_run_ws", "lacosmic_run_batch",
    "lacosmic_batch_workspace_bytes", "lacosmic_host_batch_workspace_bytes", "lacosmic_run_host_batch",
    "lacosmic_host_workspace_bytes", "lacosmic_run_host", "lacosmic_run_host_u16", "lacosmic_run_host_sparse", "lacosmic_run_host_stream_sparse", "lacosmic_estimate_gain", "lacosmic_lplus",
    "lacosmic_medfilt",
    "lacosmic_bitplane_pitch_words", "lacosmic_pack_bits", "lacosmic_unpack_bits",
    "lacosmic_dilate3", "lacosmic_masked_median", "lacosmic_strerror",
    "lacosmic_last_cuda_error", "lacosmic_last_launch_count", "lacosmic_version",
    "lacosmic_kernel_timing_enable", "lacosmic_kernel_timing_read", "lacosmic_kernel_class_name",
    "lacosmic_probe_minmax_rate", "lacosmic_stats_enable", "lacosmic_frame_stats", "lacosmic_graph_replay_enable", "lacosmic_gain_fast_path_enable", "lacosmic_gain_zone_info",
    "lacosmic_run_ex", "lacosmic_sepmed_workspace_bytes", "lacosmic_run_sepmed_compare", "lacosmic_sepmedfilt",
    "lacosmic_masked_median_bpm", "lacosmic_satstar_mask", "lacosmic_masked_median_noalloc", "lacosmic_estimate_gain_ex", "lacosmic_host_band_plan",
)
NOALLOC_MAX_WORDS = 131072       # include/lacosmic.h LACOSMIC_NOALLOC_MAX_WORDS
ERR_TOO_LARGE = -8
NUM_KERNEL_CLASSES = 9
MODE_LAZY, MODE_DENSE = 0, 1
FS_ADU, FS_NORMALISED = 0, 1


class LacosmicError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = load_library().lacosmic_strerror(code).decode()
        if code == -7:
            msg += " [cudaError %d]" % load_library().lacosmic_last_cuda_error()
        super().__init__("%s: %s (code %d)" % (where, msg, code))


class _CParams(C.Structure):
    _fields_ = [(n, C.c_float) for n in ("gain", "readnoise", "sigclip", "sigfrac", "objlim",
                                         "satlevel")] + [("niter", C.c_int32), ("mode", C.c_int32)]


class _CVariant(C.Structure):
    _fields_ = [("fsmode", C.c_int32), ("satgrow", C.c_int32), ("bpm", C.c_void_p), ("var", C.c_void_p)]


class _CDebug(C.Structure):
    _fields_ = [("iter", C.c_int32)] + [(n, C.c_void_p) for n in (
        "Lp", "N", "S", "Sp", "m3", "F", "G1", "G2", "M1", "M2", "M3", "C", "gains")]


DEBUG_F32 = ("Lp", "N", "S", "Sp", "m3", "F")
DEBUG_U8 = ("G1", "G2", "M1", "M2", "M3", "C")


@dataclass
class Params:
    """Per-frame parameters (niter/satlevel from the north_star signature)."""
    gain: float = 1.0          # 0 = not supplied: estimated at each iteration (R21)
    readnoise: float = 10.0
    sigclip: float = 4.5
    sigfrac: float = 0.3
    objlim: float = 5.0
    satlevel: float = 65535.0
    niter: int = 4
    mode: int = MODE_LAZY      # MODE_DENSE: the dense reference path (same results)

    def _c(self):
        return _CParams(self.gain, self.readnoise, self.sigclip, self.sigfrac, self.objlim,
                        self.satlevel, int(self.niter), int(self.mode))


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen liblacosmic_b200.so (built in-tree by paper_2602_17938_b200/build.py)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError(
            "liblacosmic_b200.so is missing at %s -- build it with "
            "`python -m paper_2602_17938_b200.build` (needs nvcc); there is no CPU fallback"
            % _LIB_PATH)
    L = C.CDLL(_LIB_PATH)
    vp, i, f, sz = C.c_void_p, C.c_int, C.c_float, C.c_size_t
    sig = {
        "lacosmic_run": (i, [vp, i, i, f, f, f, f, f, i, f, vp, vp, vp]),
        "lacosmic_workspace_bytes": (sz, [i, i]),
        "lacosmic_batch_workspace_bytes": (sz, [i, i, i]),
        "lacosmic_host_batch_workspace_bytes": (sz, [i, i, i]),
        "lacosmic_run_host_batch": (i, [vp, i, i, i, C.POINTER(_CParams), vp, vp, vp, sz, vp]),
        "lacosmic_run_ws": (i, [vp, i, i, C.POINTER(_CParams), vp, vp, vp, sz, vp,
                                C.POINTER(_CDebug), vp]),
        "lacosmic_run_batch": (i, [vp, i, i, i, C.POINTER(_CParams), vp, vp, vp, sz, vp, vp]),
        "lacosmic_host_workspace_bytes": (sz, [i, i]),
        "lacosmic_host_band_plan": (i, [i, i, vp, vp]),
        "lacosmic_run_host": (i, [vp, i, i, C.POINTER(_CParams), vp, vp, vp, sz, vp]),
        "lacosmic_run_host_u16": (i, [vp, i, i, C.POINTER(_CParams), vp, vp, vp, sz, vp]),
        "lacosmic_run_host_sparse": (i, [vp, i, i, C.POINTER(_CParams), vp, vp, vp, vp, i, vp, sz, vp]),
        "lacosmic_run_host_stream_sparse": (i, [vp, i, i, i, i, C.POINTER(_CParams), vp, vp, vp, vp, i, vp, sz, vp]),
        "lacosmic_estimate_gain": (i, [vp, i, i, f, vp, vp, vp, sz, vp]),
        "lacosmic_estimate_gain_ex": (i, [vp, i, i, f, vp, vp, vp, vp, sz, vp]),
        "lacosmic_lplus": (i, [vp, vp, i, i, vp]),
        "lacosmic_medfilt": (i, [vp, vp, i, i, i, vp]),
        "lacosmic_bitplane_pitch_words": (i, [i]),
        "lacosmic_pack_bits": (i, [vp, vp, i, i, vp]),
        "lacosmic_unpack_bits": (i, [vp, vp, i, i, vp]),
        "lacosmic_dilate3": (i, [vp, vp, i, i, vp]),
        "lacosmic_masked_median": (i, [vp, vp, vp, i, i, vp, sz, vp]),
        "lacosmic_strerror": (C.c_char_p, [i]),
        "lacosmic_last_cuda_error": (i, []),
        "lacosmic_last_launch_count": (i, []),
        "lacosmic_version": (C.c_char_p, []),
        "lacosmic_kernel_timing_enable": (i, [i]),
        "lacosmic_kernel_timing_read": (i, [vp, vp]),
        "lacosmic_kernel_class_name": (C.c_char_p, [i]),
        "lacosmic_probe_minmax_rate": (i, [i, vp, vp]),
        "lacosmic_stats_enable": (i, [i]),
        "lacosmic_gain_fast_path_enable": (i, [i]),
        "lacosmic_gain_zone_info": (i, [vp, i, i, vp, vp]),
        "lacosmic_graph_replay_enable": (i, [i]),
        "lacosmic_frame_stats": (i, [vp, i, i, vp, vp]),
        "lacosmic_run_ex": (i, [vp, i, i, C.POINTER(_CParams), C.POINTER(_CVariant), vp, vp, vp, sz, vp,
                                C.POINTER(_CDebug), vp]),
        "lacosmic_sepmed_workspace_bytes": (sz, [i, i]),
        "lacosmic_run_sepmed_compare": (i, [vp, i, i, C.POINTER(_CParams), vp, vp, vp, sz, vp, C.POINTER(_CDebug), vp]),
        "lacosmic_sepmedfilt": (i, [vp, vp, vp, i, i, i, vp]),
        "lacosmic_masked_median_bpm": (i, [vp, vp, vp, vp, i, i, vp, sz, vp]),
        "lacosmic_satstar_mask": (i, [vp, i, i, f, i, vp, vp, sz, vp]),
        "lacosmic_masked_median_noalloc": (i, [vp, vp, vp, vp, i, i, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)      # AttributeError if the header and the library disagree
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


# ----------------------------------------------------------------------------- marshalling helpers
def _torch():
    import torch
    return torch


def _dev(t, dtype, name, shape=None):
    torch = _torch()
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA torch tensor" % name)
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be contiguous %s" % (name, dtype))
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError("%s has shape %s, expected %s" % (name, tuple(t.shape), tuple(shape)))
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        return _torch().cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def _scratch_on(t, stream):
    """Scratch this module allocated itself is dropped when the wrapper returns, while the work enqueued on `stream`
    still uses it.  The caching allocator only orders reuse against the stream a block was allocated on (torch's
    current stream); for any other stream the block must be recorded on it, or it can be handed out again while
    the kernels still run."""
    if stream is None:
        return t
    torch = _torch()
    st = stream if isinstance(stream, torch.cuda.Stream) else torch.cuda.ExternalStream(int(stream), device=t.device)
    t.record_stream(st)
    return t


def _on_device(fn):
    """Host-buffer entry points take device=...: make it the current device for the call (the library works on the
    current device, and stream=None means that device's current stream).  `device` may be given by keyword or by
    position; it is resolved against the wrapped function's own signature."""
    import inspect
    sig = inspect.signature(fn)

    @functools.wraps(fn)
    def wrapped(*args, **kw):
        bound = sig.bind(*args, **kw)
        bound.apply_defaults()
        with _torch().cuda.device(bound.arguments["device"]):
            return fn(*bound.args, **bound.kwargs)
    return wrapped


def _check(rc, where):
    if rc != 0:
        raise LacosmicError(rc, where)


def _params(p=None, **kw):
    if p is None:
        p = Params(**kw)
    elif kw:
        raise TypeError("give either a Params object or keyword parameters")
    return p


def _workspace(h, w, like, host=False):
    torch = _torch()
    n = lacosmic_host_workspace_bytes(h, w) if host else lacosmic_workspace_bytes(h, w)
    return torch.empty(n, dtype=torch.uint8, device=like)


# ----------------------------------------------------------------------------- the whole path
def lacosmic_workspace_bytes(h, w):
    return int(load_library().lacosmic_workspace_bytes(int(h), int(w)))


def lacosmic_batch_workspace_bytes(h, w, concurrency):
    return int(load_library().lacosmic_batch_workspace_bytes(int(h), int(w), int(concurrency)))


def lacosmic_host_workspace_bytes(h, w):
    return int(load_library().lacosmic_host_workspace_bytes(int(h), int(w)))


def lacosmic_host_band_plan(h, w):
    """[(row_end, tile_rows)] per band of the banded H2D copy of the single-frame host calls ([] = one piece)."""
    re, up = (C.c_int32 * 8)(), (C.c_int32 * 8)()
    n = load_library().lacosmic_host_band_plan(int(h), int(w), re, up)
    if n < 0:
        raise LacosmicError(n, "lacosmic_host_band_plan")
    return [(int(re[b]), int(up[b])) for b in range(n)]


def lacosmic_run(img, gain=1.0, readnoise=10.0, sigclip=4.5, sigfrac=0.3, objlim=5.0, niter=4,
                 satlevel=65535.0, mask_out=None, clean_out=None, stream=None):
    """North-star call: returns (mask_out uint8 [h][w], clean_out fp32 [h][w])."""
    torch = _torch()
    L = load_library()
    if img.dim() != 2:
        raise ValueError("img must be [h][w]")
    h, w = img.shape
    ip = _dev(img, torch.float32, "img")
    if mask_out is None:
        mask_out = torch.empty((h, w), dtype=torch.uint8, device=img.device)
    if clean_out is None:
        clean_out = torch.empty_like(img)
    rc = L.lacosmic_run(ip, h, w, gain, readnoise, sigclip, sigfrac, objlim, int(niter), satlevel,
                        _dev(mask_out, torch.uint8, "mask_out", (h, w)),
                        _dev(clean_out, torch.float32, "clean_out", (h, w)), _stream(stream))
    _check(rc, "lacosmic_run")
    return mask_out, clean_out


def lacosmic_run_ws(img, params=None, mask_out=None, clean_out=None, workspace=None,
                    iter_counts=None, debug_iter=None, debug_planes=None, want_gains=False, stream=None,
                    fsmode=None, satgrow=None, bpm=None, var=None, sepmed_compare=False, **kw):
    """Timed entry point.  Returns dict(mask, clean, counts[, debug planes of iteration debug_iter][, gains =
    the gain each iteration used, when want_gains]).  Any of fsmode / satgrow / bpm (uint8 CUDA tensor) / var (float32
    CUDA tensor) given: lacosmic_run_ex with those variants (R22-R25).  sepmed_compare=True:
    lacosmic_run_sepmed_compare, the separable-median comparison path (R26)."""
    torch = _torch()
    L = load_library()
    p = _params(params, **kw)
    variant = not all(a is None for a in (fsmode, satgrow, bpm, var))
    if variant and sepmed_compare:
        raise ValueError("the separable-median comparison path takes no variants")
    if img.dim() != 2:
        raise ValueError("img must be [h][w]")
    h, w = img.shape
    ip = _dev(img, torch.float32, "img")
    if mask_out is None:
        mask_out = torch.empty((h, w), dtype=torch.uint8, device=img.device)
    if clean_out is None:
        clean_out = torch.empty_like(img)
    if workspace is None:
        nbytes = lacosmic_sepmed_workspace_bytes(h, w) if sepmed_compare else lacosmic_workspace_bytes(h, w)
        workspace = _scratch_on(torch.empty(nbytes, dtype=torch.uint8, device=img.device), stream)
    if iter_counts is None:
        iter_counts = torch.zeros(max(int(p.niter), 1), dtype=torch.int32, device=img.device)
    out = dict(mask=mask_out, clean=clean_out, counts=iter_counts)
    dbg_ref = None
    if debug_iter is not None or want_gains:
        dbg = _CDebug()
        dbg.iter = int(debug_iter) if debug_iter is not None else -1
        if debug_iter is not None:
            names = debug_planes if debug_planes is not None else DEBUG_F32 + DEBUG_U8
            for n in names:
                dt = torch.float32 if n in DEBUG_F32 else torch.uint8
                out[n] = torch.zeros((h, w), dtype=dt, device=img.device)
                setattr(dbg, n, out[n].data_ptr())
        if want_gains:
            out["gains"] = torch.zeros(max(int(p.niter), 1), dtype=torch.float32, device=img.device)
            dbg.gains = out["gains"].data_ptr()
        dbg_ref = C.byref(dbg)
    cp = p._c()
    tail = (_dev(mask_out, torch.uint8, "mask_out", (h, w)), _dev(clean_out, torch.float32, "clean_out", (h, w)),
            _dev(workspace, torch.uint8, "workspace"), workspace.numel(),
            _dev(iter_counts, torch.int32, "iter_counts"), dbg_ref, _stream(stream))
    if sepmed_compare:
        _check(L.lacosmic_run_sepmed_compare(ip, h, w, C.byref(cp), *tail), "lacosmic_run_sepmed_compare")
    elif variant:
        cv = _CVariant(int(fsmode or 0), -1 if satgrow is None else int(satgrow),
                       None if bpm is None else _dev(bpm, torch.uint8, "bpm", (h, w)),
                       None if var is None else _dev(var, torch.float32, "var", (h, w)))
        _check(L.lacosmic_run_ex(ip, h, w, C.byref(cp), C.byref(cv), *tail), "lacosmic_run_ex")
    else:
        _check(L.lacosmic_run_ws(ip, h, w, C.byref(cp), *tail), "lacosmic_run_ws")
    return out


def lacosmic_run_ex(img, params=None, fsmode=FS_ADU, satgrow=-1, bpm=None, var=None, **kw):
    """lacosmic_run_ws with the variants of DESIGN.md R22-R25 (always through the lacosmic_run_ex entry point)."""
    return lacosmic_run_ws(img, params, fsmode=fsmode, satgrow=satgrow, bpm=bpm, var=var, **kw)


def lacosmic_run_sepmed_compare(img, params=None, **kw):
    """The separable-median comparison path (R26).  Not a product path."""
    return lacosmic_run_ws(img, params, sepmed_compare=True, **kw)


def lacosmic_sepmed_workspace_bytes(h, w):
    return int(load_library().lacosmic_sepmed_workspace_bytes(int(h), int(w)))


def lacosmic_sepmedfilt(img, k, out=None, stream=None):
    torch = _torch()
    h, w = img.shape
    if out is None:
        out = torch.empty_like(img)
    tmp = _scratch_on(torch.empty_like(img), stream)
    _check(load_library().lacosmic_sepmedfilt(_dev(img, torch.float32, "img"), _dev(out, torch.float32, "out", (h, w)),
                                              tmp.data_ptr(), h, w, int(k), _stream(stream)), "lacosmic_sepmedfilt")
    return out


def lacosmic_satstar_mask(img, satlevel=65535.0, grow=0, workspace=None, stream=None):
    """R25 alone: uint8 [h][w], 1 on dil3^grow(med5(img) >= satlevel)."""
    torch = _torch()
    h, w = img.shape
    out = torch.empty((h, w), dtype=torch.uint8, device=img.device)
    if workspace is None:
        workspace = _scratch_on(_workspace(h, w, img.device), stream)
    _check(load_library().lacosmic_satstar_mask(_dev(img, torch.float32, "img"), h, w, float(satlevel), int(grow),
                                                out.data_ptr(), _dev(workspace, torch.uint8, "workspace"),
                                                workspace.numel(), _stream(stream)), "lacosmic_satstar_mask")
    return out


def lacosmic_run_batch(imgs, params, masks_out=None, cleans_out=None, workspace=None,
                       iter_counts=None, stream=None, concurrency=1):
    """imgs [n][h][w]; params: list of n Params.  Returns dict(mask, clean, counts [n][MAX_NITER]).
    `concurrency` sizes the workspace this call allocates when none is given (frames in flight)."""
    torch = _torch()
    L = load_library()
    if imgs.dim() != 3:
        raise ValueError("imgs must be [n][h][w]")
    n, h, w = imgs.shape
    if len(params) != n:
        raise ValueError("need one Params per frame")
    arr = (_CParams * max(n, 1))(*[p._c() for p in params])
    if masks_out is None:
        masks_out = torch.empty((n, h, w), dtype=torch.uint8, device=imgs.device)
    if cleans_out is None:
        cleans_out = torch.empty_like(imgs)
    if workspace is None:
        workspace = _scratch_on(torch.empty(max(lacosmic_batch_workspace_bytes(h, w, max(1, concurrency)), 256),
                                            dtype=torch.uint8, device=imgs.device), stream)
    if iter_counts is None:
        iter_counts = torch.zeros((max(n, 1), MAX_NITER), dtype=torch.int32, device=imgs.device)
    rc = L.lacosmic_run_batch(_dev(imgs, torch.float32, "imgs"), n, h, w, arr,
                              _dev(masks_out, torch.uint8, "masks_out", (n, h, w)),
                              _dev(cleans_out, torch.float32, "cleans_out", (n, h, w)),
                              _dev(workspace, torch.uint8, "workspace"), workspace.numel(),
                              _dev(iter_counts, torch.int32, "iter_counts"), _stream(stream))
    _check(rc, "lacosmic_run_batch")
    return dict(mask=masks_out, clean=cleans_out, counts=iter_counts)


@_on_device
def lacosmic_run_host(img_host, params=None, mask_out_host=None, clean_out_host=None,
                      dev_workspace=None, device="cuda:0", stream=None, **kw):
    """End-to-end call with HOST (ideally pinned) torch CPU tensors; copies are part of the call.  img_host is
    float32, or uint16 (the detector's raw counts: copied as 2 bytes per pixel, widened on the device)."""
    torch = _torch()
    L = load_library()
    p = _params(params, **kw)
    if (not isinstance(img_host, torch.Tensor) or img_host.is_cuda or not img_host.is_contiguous()
            or img_host.dtype not in (torch.float32, torch.uint16)):
        raise TypeError("img_host must be a contiguous CPU float32 or uint16 tensor")
    h, w = img_host.shape
    if mask_out_host is None:
        mask_out_host = torch.empty((h, w), dtype=torch.uint8).pin_memory()
    if clean_out_host is None:
        clean_out_host = torch.empty((h, w), dtype=torch.float32).pin_memory()
    if dev_workspace is None:
        dev_workspace = _scratch_on(_workspace(h, w, device, host=True), stream)
    cp = p._c()
    fn = L.lacosmic_run_host_u16 if img_host.dtype == torch.uint16 else L.lacosmic_run_host
    rc = fn(img_host.data_ptr(), h, w, C.byref(cp), mask_out_host.data_ptr(),
            clean_out_host.data_ptr(), _dev(dev_workspace, torch.uint8, "dev_workspace"),
            dev_workspace.numel(), _stream(stream))
    _check(rc, "lacosmic_run_host")
    # the call has only ENQUEUED the H2D copy (on `stream`, or in bands on the library's copy stream): the result keeps
    # the input tensor referenced so that a temporary (e.g. x.pin_memory()) is not handed back to torch's host allocator,
    # and possibly reused, before the copy has read it.  The caller must still not WRITE img_host before synchronising.
    return dict(mask=mask_out_host, clean=clean_out_host, _img_host=img_host)


@_on_device
def lacosmic_run_host_sparse(img_host, params=None, capacity=None, out=None, dev_workspace=None,
                             device="cuda:0", stream=None, **kw):
    """Sparse results (host tensors): dict(maskbits int32 [h][pitch], idx int32 [capacity], val float32
    [capacity], count int32 [1]).  capacity defaults to 1/16 of the frame.  Pass `out` (a previous result) to
    reuse its pinned buffers."""
    torch = _torch()
    L = load_library()
    p = _params(params, **kw)
    if (not isinstance(img_host, torch.Tensor) or img_host.is_cuda or not img_host.is_contiguous()
            or img_host.dtype != torch.float32):
        raise TypeError("img_host must be a contiguous CPU float32 tensor")
    h, w = img_host.shape
    pitch = lacosmic_bitplane_pitch_words(w)
    if out is None:
        cap = int(capacity) if capacity is not None else max(1, (h * w) // 16)
        out = dict(maskbits=torch.empty((h, pitch), dtype=torch.int32).pin_memory(),
                   idx=torch.empty(max(cap, 1), dtype=torch.int32).pin_memory(),
                   val=torch.empty(max(cap, 1), dtype=torch.float32).pin_memory(),
                   count=torch.zeros(1, dtype=torch.int32).pin_memory(), capacity=cap)
    if dev_workspace is None:
        dev_workspace = _scratch_on(_workspace(h, w, device, host=True), stream)
    cp = p._c()
    rc = L.lacosmic_run_host_sparse(img_host.data_ptr(), h, w, C.byref(cp), out["maskbits"].data_ptr(),
                                    out["idx"].data_ptr(), out["val"].data_ptr(), out["count"].data_ptr(),
                                    int(out["capacity"]), _dev(dev_workspace, torch.uint8, "dev_workspace"),
                                    dev_workspace.numel(), _stream(stream))
    _check(rc, "lacosmic_run_host_sparse")
    out["_img_host"] = img_host          # stays referenced until the caller drops the result (see lacosmic_run_host)
    return out


@_on_device
def lacosmic_run_host_stream_sparse(imgs_host, params, capacity=None, out=None, dev_workspace=None,
                                    device="cuda:0", stream=None, concurrency=3):
    """Stream of host frames [n][h][w] (float32 or uint16), sparse results per frame: dict(maskbits int32
    [n][h][pitch], idx int32 [n][capacity], val float32 [n][capacity], count int32 [n])."""
    torch = _torch()
    L = load_library()
    if (not isinstance(imgs_host, torch.Tensor) or imgs_host.is_cuda or not imgs_host.is_contiguous()
            or imgs_host.dim() != 3 or imgs_host.dtype not in (torch.float32, torch.uint16)):
        raise TypeError("imgs_host must be a contiguous CPU float32 or uint16 tensor [n][h][w]")
    n, h, w = imgs_host.shape
    if len(params) != n:
        raise ValueError("need one Params per frame")
    arr = (_CParams * max(n, 1))(*[p._c() for p in params])
    pitch = lacosmic_bitplane_pitch_words(w)
    if out is None:
        cap = int(capacity) if capacity is not None else max(1, (h * w) // 16)
        out = dict(maskbits=torch.empty((n, h, pitch), dtype=torch.int32).pin_memory(),
                   idx=torch.empty((n, max(cap, 1)), dtype=torch.int32).pin_memory(),
                   val=torch.empty((n, max(cap, 1)), dtype=torch.float32).pin_memory(),
                   count=torch.zeros(n, dtype=torch.int32).pin_memory(), capacity=cap)
    if dev_workspace is None:
        dev_workspace = _scratch_on(torch.empty(max(lacosmic_host_batch_workspace_bytes(h, w, max(1, concurrency)), 256),
                                                dtype=torch.uint8, device=device), stream)
    rc = L.lacosmic_run_host_stream_sparse(imgs_host.data_ptr(), int(imgs_host.dtype == torch.uint16), n, h, w, arr,
                                           out["maskbits"].data_ptr(), out["idx"].data_ptr(), out["val"].data_ptr(),
                                           out["count"].data_ptr(), int(out["capacity"]),
                                           _dev(dev_workspace, torch.uint8, "dev_workspace"), dev_workspace.numel(),
                                           _stream(stream))
    _check(rc, "lacosmic_run_host_stream_sparse")
    out["_img_host"] = imgs_host
    return out


def lacosmic_clean(image, gain=1.0, readnoise=10.0, sigclip=4.5, sigfrac=0.3, objlim=5.0, niter=4,
                   satlevel=65535.0, device="cuda:0", fsmode=FS_ADU, satgrow=None, bpm=None, var=None):
    """The user-level entry point of the paper (one call with objlim, sigfrac, sigclip and
    optional gain / readnoise): a 2-D numpy array (float32, or the detector's uint16 counts) in, (mask bool
    [h][w], cleaned float32 [h][w]) numpy arrays out.  gain=0 (or None): estimated at each iteration.  Every
    step runs in the CUDA library; this wrapper only stages buffers.

    Fidelity note.  The default object test is the north-star text's (R7): L+/F > objlim with the fine
    structure F in ADU.  van Dokkum's original form, which dfcosmic ports, compares S' with the fine structure in units
    of the noise: fsmode=FS_NORMALISED (R22) selects it -- there the same objlim is about twice as strict (S'/Fn is
    (L+/F)/2 where med5(S) = 0), so masks differ between the two settings.  satgrow=k protects (near-)saturated star
    cores (R25), bpm / var are an input bad-pixel mask and a variance plane (R23, R24).  None of these readings could be
    checked against dfcosmic's code or the IRAF masks (not available): expect differences in detail on real data."""
    import numpy as np
    torch = _torch()
    a = np.ascontiguousarray(image)
    if a.ndim != 2:
        raise ValueError("image must be 2-D")
    if a.dtype != np.uint16:
        a = a.astype(np.float32, copy=False)
    p = Params(gain=0.0 if gain is None else float(gain), readnoise=readnoise, sigclip=sigclip, sigfrac=sigfrac,
               objlim=objlim, satlevel=satlevel, niter=niter)
    variant = fsmode != FS_ADU or satgrow is not None or bpm is not None or var is not None
    with torch.cuda.device(device):
        if variant:      # the variants take device planes (lacosmic_run_ex)
            dev = torch.device(device)
            img = torch.from_numpy(a.astype(np.float32, copy=False)).to(dev)
            kw = dict(fsmode=fsmode, satgrow=-1 if satgrow is None else satgrow)
            if bpm is not None:
                kw["bpm"] = torch.from_numpy(np.ascontiguousarray(bpm).astype(np.uint8)).to(dev)
            if var is not None:
                kw["var"] = torch.from_numpy(np.ascontiguousarray(var, dtype=np.float32)).to(dev)
            r = lacosmic_run_ex(img, p, **kw)
            torch.cuda.current_stream().synchronize()
            return r["mask"].cpu().numpy().astype(bool), r["clean"].cpu().numpy()
        pinned = torch.from_numpy(a).pin_memory()          # stays referenced until the copy has completed
        r = lacosmic_run_host(pinned, p, device=device)
        torch.cuda.current_stream().synchronize()
    del pinned
    return r["mask"].numpy().astype(bool), r["clean"].numpy()


def lacosmic_host_batch_workspace_bytes(h, w, concurrency):
    return int(load_library().lacosmic_host_batch_workspace_bytes(int(h), int(w), int(concurrency)))


@_on_device
def lacosmic_run_host_batch(imgs_host, params, masks_host=None, cleans_host=None, dev_workspace=None,
                            device="cuda:0", stream=None, concurrency=3):
    """Stream of frames in HOST (ideally pinned) tensors [n][h][w]; params: list of n Params.  `concurrency`
    staging slots are in flight (sizes the device scratch this call allocates when none is given)."""
    torch = _torch()
    L = load_library()
    if (not isinstance(imgs_host, torch.Tensor) or imgs_host.is_cuda or imgs_host.dtype != torch.float32
            or not imgs_host.is_contiguous() or imgs_host.dim() != 3):
        raise TypeError("imgs_host must be a contiguous CPU float32 tensor [n][h][w]")
    n, h, w = imgs_host.shape
    if len(params) != n:
        raise ValueError("need one Params per frame")
    arr = (_CParams * max(n, 1))(*[p._c() for p in params])
    if masks_host is None:
        masks_host = torch.empty((n, h, w), dtype=torch.uint8).pin_memory()
    if cleans_host is None:
        cleans_host = torch.empty((n, h, w), dtype=torch.float32).pin_memory()
    if dev_workspace is None:
        dev_workspace = _scratch_on(torch.empty(max(lacosmic_host_batch_workspace_bytes(h, w, max(1, concurrency)), 256),
                                                dtype=torch.uint8, device=device), stream)
    rc = L.lacosmic_run_host_batch(imgs_host.data_ptr(), n, h, w, arr, masks_host.data_ptr(),
                                   cleans_host.data_ptr(), _dev(dev_workspace, torch.uint8, "dev_workspace"),
                                   dev_workspace.numel(), _stream(stream))
    _check(rc, "lacosmic_run_host_batch")
    return dict(mask=masks_host, clean=cleans_host, _img_host=imgs_host)


# ----------------------------------------------------------------------------- single steps
def lacosmic_gain_zone_info(workspace, h, w, stream=None):
    """Diagnostic: the plan of the last gain estimate run in `workspace` as 40 int32 words (include/lacosmic.h)."""
    import numpy as np
    torch = _torch()
    buf = np.zeros(40, np.int32)
    _check(load_library().lacosmic_gain_zone_info(_dev(workspace, torch.uint8, "workspace"), int(h), int(w),
                                                  buf.ctypes.data, _stream(stream)), "lacosmic_gain_zone_info")
    return buf


def lacosmic_gain_fast_path_enable(enable=True):
    _check(load_library().lacosmic_gain_fast_path_enable(1 if enable else 0), "lacosmic_gain_fast_path_enable")


def lacosmic_estimate_gain(img, readnoise=0.0, workspace=None, stream=None, want_path=False):
    """R21 alone.  Returns (gain: device float tensor [1], stats: device float tensor [6] = c, s, lo, hi, kept, mt);
    with want_path also a device float tensor [1]: 1 if the clipping rounds ran on the zone lists, 0 if on the plane."""
    torch = _torch()
    h, w = img.shape
    if workspace is None:
        workspace = _scratch_on(_workspace(h, w, img.device), stream)
    gain = torch.zeros(1, dtype=torch.float32, device=img.device)
    stats = torch.zeros(6, dtype=torch.float32, device=img.device)
    args = (_dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream))
    if want_path:
        path = torch.zeros(1, dtype=torch.float32, device=img.device)
        _check(load_library().lacosmic_estimate_gain_ex(
            _dev(img, torch.float32, "img"), h, w, float(readnoise), gain.data_ptr(), stats.data_ptr(), path.data_ptr(),
            *args), "lacosmic_estimate_gain_ex")
        return gain, stats, path
    _check(load_library().lacosmic_estimate_gain(
        _dev(img, torch.float32, "img"), h, w, float(readnoise), gain.data_ptr(), stats.data_ptr(), *args),
        "lacosmic_estimate_gain")
    return gain, stats


def lacosmic_lplus(img, out=None, stream=None):
    torch = _torch()
    h, w = img.shape
    if out is None:
        out = torch.empty_like(img)
    _check(load_library().lacosmic_lplus(_dev(img, torch.float32, "img"),
                                         _dev(out, torch.float32, "out", (h, w)), h, w,
                                         _stream(stream)), "lacosmic_lplus")
    return out


def lacosmic_medfilt(img, k, out=None, stream=None):
    torch = _torch()
    h, w = img.shape
    if out is None:
        out = torch.empty_like(img)
    _check(load_library().lacosmic_medfilt(_dev(img, torch.float32, "img"),
                                           _dev(out, torch.float32, "out", (h, w)), h, w, int(k),
                                           _stream(stream)), "lacosmic_medfilt")
    return out


def lacosmic_bitplane_pitch_words(w):
    return int(load_library().lacosmic_bitplane_pitch_words(int(w)))


def lacosmic_pack_bits(mask_u8, stream=None):
    torch = _torch()
    h, w = mask_u8.shape
    bits = torch.empty((h, lacosmic_bitplane_pitch_words(w)), dtype=torch.int32, device=mask_u8.device)
    _check(load_library().lacosmic_pack_bits(_dev(mask_u8, torch.uint8, "mask_u8"), bits.data_ptr(),
                                             h, w, _stream(stream)), "lacosmic_pack_bits")
    return bits


def lacosmic_unpack_bits(bits, h, w, stream=None):
    torch = _torch()
    out = torch.empty((h, w), dtype=torch.uint8, device=bits.device)
    _check(load_library().lacosmic_unpack_bits(
        _dev(bits, torch.int32, "bits", (h, lacosmic_bitplane_pitch_words(w))), out.data_ptr(), h, w,
        _stream(stream)), "lacosmic_unpack_bits")
    return out


def lacosmic_dilate3(bits, h, w, stream=None):
    """bits: int32 [h][pitch] bit-plane (LSB = lowest x).  Returns the dilated bit-plane."""
    torch = _torch()
    out = torch.empty_like(bits)
    _check(load_library().lacosmic_dilate3(
        _dev(bits, torch.int32, "bits", (h, lacosmic_bitplane_pitch_words(w))), out.data_ptr(), h, w,
        _stream(stream)), "lacosmic_dilate3")
    return out


def lacosmic_masked_median(img, mask_u8, out=None, workspace=None, stream=None, bpm=None):
    """Step (7).  bpm (uint8 CUDA tensor): bad pixels removed from the donors (R23, lacosmic_masked_median_bpm)."""
    torch = _torch()
    h, w = img.shape
    if out is None:
        out = torch.empty_like(img)
    if workspace is None:
        workspace = _scratch_on(_workspace(h, w, img.device), stream)
    L = load_library()
    args = (_dev(out, torch.float32, "out", (h, w)), h, w, _dev(workspace, torch.uint8, "workspace"),
            workspace.numel(), _stream(stream))
    if bpm is None:
        _check(L.lacosmic_masked_median(_dev(img, torch.float32, "img"), _dev(mask_u8, torch.uint8, "mask_u8", (h, w)),
                                        *args), "lacosmic_masked_median")
    else:
        _check(L.lacosmic_masked_median_bpm(_dev(img, torch.float32, "img"), _dev(mask_u8, torch.uint8, "mask_u8", (h, w)),
                                            _dev(bpm, torch.uint8, "bpm", (h, w)), *args), "lacosmic_masked_median_bpm")
    return out


lacosmic_masked_median_bpm = lacosmic_masked_median


def lacosmic_masked_median_noalloc(img, mask_u8, out, bpm=None, stream=None):
    """Step (7) for a caller that cannot allocate device memory (a plug-in inside an application that owns the GPU
    memory pool, a real-time loop that must stay out of the allocator, a process at its memory budget): the scratch
    is a fixed array inside the library instead of a workspace.  `out` is required -- this wrapper allocates nothing
    either.  Same result as lacosmic_masked_median(img, mask_u8, bpm=bpm), bit for bit.

    Limit: h * ceil(w / 32) <= NOALLOC_MAX_WORDS (any frame up to 2048 x 2048); larger frames raise LacosmicError with
    code ERR_TOO_LARGE and leave `out` untouched.  All calls on one GPU share the one array: calls ordered on the GPU
    (same stream) are fine, calls that may overlap on the GPU race.  The first call on a device looks the array's
    address up; make it during set-up."""
    torch = _torch()
    h, w = img.shape
    rc = load_library().lacosmic_masked_median_noalloc(
        _dev(img, torch.float32, "img"), _dev(mask_u8, torch.uint8, "mask_u8", (h, w)),
        None if bpm is None else _dev(bpm, torch.uint8, "bpm", (h, w)),
        _dev(out, torch.float32, "out", (h, w)), h, w, _stream(stream))
    _check(rc, "lacosmic_masked_median_noalloc")
    return out


def lacosmic_strerror(code):
    return load_library().lacosmic_strerror(int(code)).decode()


def lacosmic_last_launch_count():
    return int(load_library().lacosmic_last_launch_count())


def lacosmic_version():
    return load_library().lacosmic_version().decode()


def lacosmic_kernel_timing_enable(enable=True):
    _check(load_library().lacosmic_kernel_timing_enable(1 if enable else 0),
           "lacosmic_kernel_timing_enable")


def lacosmic_probe_minmax_rate(kind=0, stream=None):
    """Measured fp32 min/max issue rate of the current device in instructions/s (kind 0: FMNMX, 1: FMNMX3).
    Synchronises the stream."""
    out = C.c_double(0.0)
    _check(load_library().lacosmic_probe_minmax_rate(int(kind), C.byref(out), _stream(stream)),
           "lacosmic_probe_minmax_rate")
    return float(out.value)


def lacosmic_stats_enable(enable=True):
    _check(load_library().lacosmic_stats_enable(1 if enable else 0), "lacosmic_stats_enable")


def lacosmic_graph_replay_enable(enable=True):
    """Switch the CUDA-graph replay of repeated identical lacosmic_run_ws calls on or off (process-wide; on by default)."""
    _check(load_library().lacosmic_graph_replay_enable(1 if enable else 0), "lacosmic_graph_replay_enable")


def lacosmic_frame_stats(workspace, h, w, stream=None):
    """{name: [per-iteration int]} of the last frame that ran in `workspace` (synchronises the stream)."""
    torch = _torch()
    buf = (C.c_int32 * (5 * MAX_NITER))()
    _check(load_library().lacosmic_frame_stats(_dev(workspace, torch.uint8, "workspace"), int(h), int(w), buf,
                                               _stream(stream)), "lacosmic_frame_stats")
    names = ("new", "candidates", "quads", "replaced", "fine_tests")
    return {n: [int(buf[r * MAX_NITER + t]) for t in range(MAX_NITER)] for r, n in enumerate(names)}


def lacosmic_kernel_timing_read():
    """{class name: (summed ms, spans)} since the last read; synchronise the stream first."""
    L = load_library()
    ms = (C.c_float * NUM_KERNEL_CLASSES)()
    n = (C.c_int32 * NUM_KERNEL_CLASSES)()
    _check(L.lacosmic_kernel_timing_read(ms, n), "lacosmic_kernel_timing_read")
    return {L.lacosmic_kernel_class_name(c).decode(): (float(ms[c]), int(n[c]))
            for c in range(NUM_KERNEL_CLASSES)}
