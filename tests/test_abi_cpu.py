"""CPU-side checks of the C-ABI boundary (-m "not gpu"): the library builds and loads, exports every
symbol include/lacosmic.h declares, and rejects bad arguments before touching the GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2602_17938_b200 import build, binding
    build.build()
    return binding.load_library()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "lacosmic.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lacosmic_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(L):
    names = _declared_functions()
    assert len(names) >= 15
    for n in names:
        assert hasattr(L, n), "include/lacosmic.h declares %s but the library does not export it" % n


def test_binding_lists_every_declared_symbol():
    from paper_2602_17938_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_functions()


def test_params_struct_layout():
    from paper_2602_17938_b200 import binding
    assert C.sizeof(binding._CParams) == 32          # 6 floats + 2 int32, no padding
    assert C.sizeof(binding._CDebug) == 8 + 13 * 8


def test_workspace_sizes(L):
    assert L.lacosmic_workspace_bytes(0, 5) == 0
    assert L.lacosmic_workspace_bytes(5, -1) == 0
    assert L.lacosmic_workspace_bytes(65536, 65536) == 0          # h*w >= 2^31
    n = L.lacosmic_workspace_bytes(4000, 6500)
    assert 2 * 4000 * 6500 * 4 < n < 3 * 4000 * 6500 * 4
    assert L.lacosmic_host_workspace_bytes(4000, 6500) > n + 2 * 4000 * 6500 * 4
    assert L.lacosmic_bitplane_pitch_words(6500) == 204
    assert L.lacosmic_bitplane_pitch_words(32) == 1 and L.lacosmic_bitplane_pitch_words(33) == 2


def test_argument_errors_without_gpu(L):
    """Validation happens before any CUDA call, so these run on a machine with no GPU."""
    from paper_2602_17938_b200.binding import _CParams
    ok = _CParams(1.0, 10.0, 4.5, 0.3, 5.0, 65535.0, 4, 0)
    fake = lambda a: C.c_void_p(a)                     # never dereferenced: checks fail first
    img, mask, clean, ws = 0x10000000, 0x20000000, 0x30000000, 0x40000000
    need = L.lacosmic_workspace_bytes(64, 64)
    run = lambda p=ok, i=img, m=mask, c=clean, w_=ws, nb=need, h=64, w=64: L.lacosmic_run_ws(
        fake(i), h, w, C.byref(p), fake(m), fake(c), fake(w_), nb, None, None, None)
    assert run(i=0) == -1 and run(m=0) == -1 and run(c=0) == -1 and run(w_=0) == -1
    assert run(h=0) == -2 and run(w=0) == -2
    assert run(i=img + 4) == -4 and run(w_=ws + 16) == -4
    assert run(c=img) == -5 and run(m=img + 100) == -5 and run(w_=img) == -5
    assert run(nb=need - 1) == -6
    bads = [dict(gain=-1.0), dict(gain=float("nan")), dict(readnoise=-1.0), dict(sigclip=0.0),
            dict(sigfrac=0.0), dict(sigfrac=1.5), dict(objlim=-0.1), dict(niter=-1), dict(niter=65),
            dict(satlevel=float("nan")), dict(sigclip=float("inf")), dict(mode=2), dict(mode=-1)]
    for b in bads:
        kw = dict(gain=1.0, readnoise=10.0, sigclip=4.5, sigfrac=0.3, objlim=5.0, satlevel=65535.0,
                  niter=4, mode=0)
        kw.update(b)
        assert run(p=_CParams(*[kw[k] for k in ("gain", "readnoise", "sigclip", "sigfrac", "objlim",
                                                 "satlevel", "niter", "mode")])) == -3, b
    assert L.lacosmic_medfilt(fake(img), fake(clean), 8, 8, 4, None) == -3
    assert L.lacosmic_medfilt(fake(img), fake(img), 8, 8, 3, None) == -5
    assert L.lacosmic_lplus(None, fake(clean), 8, 8, None) == -1
    assert L.lacosmic_strerror(-3) == b"invalid parameter"
    assert L.lacosmic_version().startswith(b"lacosmic-b200")


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    from paper_2602_17938_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.lacosmic_workspace_bytes(8, 8)


def test_product_path_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2602_17938_b200")
    for dp, _, fns in os.walk(pkg):
        for fn in fns:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, fn)).read()
                assert "lacosmic_oracle" not in txt, fn
                assert not re.search(r"^\s*(import|from)\s+oracle", txt, flags=re.M), fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            code = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2602_17938_b200", code, flags=re.M), fn


def test_band_plan_never_releases_a_tile_row_early(L):
    """The banded H2D copy of the single-frame host calls (include/lacosmic.h, lacosmic_host_band_plan): for EVERY height
    the rows of tiles released after band b read only rows that bands 0..b have delivered.  A row of tiles j of the first
    pass reads input rows [32 j - 2, 32 (j + 1) + 2) (LACOSMIC_HOST_TILE_ROWS / _MARGIN: the TMA box of k_noise_S_tma).
    The GPU tests (tests/test_gpu_host_banded.py) poison the staging plane, but a read that is early by a few rows is
    usually hidden by the copy engine outrunning the kernel; this check does not depend on timing."""
    TH, MY, NB = 32, 2, 8
    re, up = (C.c_int32 * NB)(), (C.c_int32 * NB)()
    for w in (4, 8, 6500, 6504):
        for h in list(range(1, 2200)) + [3999, 4000, 4001, 4097, 65535]:
            if h * w >= 2 ** 31:
                continue
            n = L.lacosmic_host_band_plan(h, w, re, up)
            nty = (h + TH - 1) // TH
            if nty < 4 * NB:
                assert n == 0, (h, w)
                continue
            assert n == NB, (h, w)
            ends, rows = [re[b] for b in range(n)], [up[b] for b in range(n)]
            assert ends == sorted(ends) and ends[-1] == h and ends[0] > 0, (h, w, ends)
            assert rows == sorted(rows) and rows[-1] == nty, (h, w, rows)
            for b in range(n):
                if ends[b] < h:
                    assert TH * rows[b] + MY <= ends[b], "tile row %d released before row %d arrived (h=%d)" % (
                        rows[b] - 1, TH * rows[b] + MY - 1, h)
                    # and not needlessly late: one more row of tiles would not have been fed (or an earlier band already
                    # released it)
                    assert TH * (rows[b] + 1) + MY > ends[b] or rows[b] == nty, (h, w, b)
                else:
                    assert rows[b] == nty
    assert L.lacosmic_host_band_plan(4000, 6501, re, up) == 0          # no TMA path for this pitch: one piece
    assert L.lacosmic_host_band_plan(0, 8, re, up) == -2 and L.lacosmic_host_band_plan(8, 8, None, up) == -1


def test_variant_inputs_may_not_alias_the_workspace(L):
    from paper_2602_17938_b200.binding import _CParams, _CVariant
    ok = _CParams(1.0, 10.0, 4.5, 0.3, 5.0, 65535.0, 4, 0)
    fake = lambda a: C.c_void_p(a)
    img, mask, clean, ws = 0x10000000, 0x20000000, 0x30000000, 0x40000000
    need = L.lacosmic_workspace_bytes(64, 64)
    run = lambda v: L.lacosmic_run_ex(fake(img), 64, 64, C.byref(ok), C.byref(v), fake(mask), fake(clean), fake(ws),
                                      need, None, None, None)
    assert run(_CVariant(0, -1, ws + 512, None)) == -5                 # bpm inside the workspace
    assert run(_CVariant(0, -1, None, ws + need - 16)) == -5           # var overlapping its end
    assert run(_CVariant(0, -1, clean + 4, None)) == -5 and run(_CVariant(0, -1, None, mask)) == -5
    assert run(_CVariant(2, -1, None, None)) == -3                     # (unknown fsmode: still a parameter error)
