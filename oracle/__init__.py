"""ctypes front end of the float64 CPU oracle (oracle/mred_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2008_11486_b200 and the CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from types import SimpleNamespace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mred_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

MEDIAN, MEAN, SIGCLIP, MINMAX, MEDCLIP = 0, 1, 2, 3, 4
SPLINE, BILINEAR, NEAREST = 0, 1, 2
PARABOLA, GAUSSIAN = 0, 1


def build(force: bool = False) -> str:
    """gcc -O2 (no fast-math: IEEE evaluation order is part of the oracle)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-fPIC", "-shared", "-fno-fast-math",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Geom(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("W", "H", "os_x0", "os_x1", "x0", "y0", "w", "h")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_combine_column.restype = C.c_double
    return _lib


def _geom(g):
    t = g.astuple() if hasattr(g, "astuple") else tuple(g)
    return _Geom(*[int(v) for v in t])


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def _u16(a):
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16
    return a


def _f32(a):
    a = np.ascontiguousarray(a)
    assert a.dtype == np.float32, a.dtype
    return a


def level(geom, raw):
    raw = _u16(raw)
    n = raw.shape[0]
    out = np.empty(n, dtype=np.float64)
    lib().orc_level(C.byref(_geom(geom)), _p(raw, C.c_uint16), C.c_int(n), _p(out, C.c_double))
    return out


def combine_column(v, mode, ksigma=3.0, max_iter=3):
    v = np.ascontiguousarray(v, dtype=np.float64)
    m = v.shape[0]
    keep = np.zeros(max(m, 1), dtype=np.uint8)
    cnt = C.c_int(0)
    mg = C.c_double(0.0)
    val = lib().orc_combine_column(_p(v, C.c_double), C.c_int(m), C.c_int(mode), C.c_double(ksigma),
                                   C.c_int(max_iter), _p(keep, C.c_uint8), C.byref(cnt), C.byref(mg))
    return SimpleNamespace(value=val, keep=keep[:m].astype(bool), count=cnt.value, margin=mg.value)


def build_masters(geom, bias, dark, t_dark, flat, t_flat, mode=MEDIAN, ksigma=3.0, max_iter=3):
    bias, dark, flat = _u16(bias), _u16(dark), _u16(flat)
    g = _geom(geom)
    shp = (g.h, g.w)
    o = SimpleNamespace(MB64=np.empty(shp), MD64=np.empty(shp), MF64=np.empty(shp),
                        MB=np.empty(shp, np.float32), MD=np.empty(shp, np.float32), MF=np.empty(shp, np.float32))
    rc = lib().orc_build_masters(C.byref(g), _p(bias, C.c_uint16), C.c_int(bias.shape[0]),
                                 _p(dark, C.c_uint16), C.c_int(dark.shape[0]), C.c_double(t_dark),
                                 _p(flat, C.c_uint16), C.c_int(flat.shape[0]), C.c_double(t_flat),
                                 C.c_int(mode), C.c_double(ksigma), C.c_int(max_iter),
                                 _p(o.MB64, C.c_double), _p(o.MD64, C.c_double), _p(o.MF64, C.c_double),
                                 _p(o.MB, C.c_float), _p(o.MD, C.c_float), _p(o.MF, C.c_float))
    if rc:
        raise ValueError("orc_build_masters: %d" % rc)
    return o


def calibrate(geom, raw, dark_scale, MB, MD, MF, want64=False):
    raw, MB, MD, MF = _u16(raw), _f32(MB), _f32(MD), _f32(MF)
    g = _geom(geom)
    n = raw.shape[0]
    out32 = np.empty((n, g.h, g.w), np.float32)
    out64 = np.empty((n, g.h, g.w), np.float64) if want64 else None
    lev = np.empty(n, np.float64)
    lib().orc_calibrate(C.byref(g), _p(raw, C.c_uint16), C.c_int(n), C.c_double(dark_scale),
                        _p(MB, C.c_float), _p(MD, C.c_float), _p(MF, C.c_float),
                        _p(out64, C.c_double), _p(out32, C.c_float), _p(lev, C.c_double))
    return SimpleNamespace(out=out32, out64=out64, level=lev)


def estimate_shifts(frames, ref_index=0, max_lag=32, badmask=None, peak=PARABOLA):
    frames = _f32(frames)
    n, h, w = frames.shape
    if badmask is not None:
        badmask = np.ascontiguousarray(badmask, dtype=np.uint8)
        assert badmask.shape == (h, w)
    ish = np.zeros((n, 2), np.int32)
    sh = np.zeros((n, 2), np.float64)
    rc = lib().orc_estimate_shifts_peak(_p(frames, C.c_float), C.c_int(n), C.c_int(w), C.c_int(h),
                                        C.c_int(ref_index), C.c_int(max_lag), _p(badmask, C.c_uint8), C.c_int(peak),
                                        _p(ish, C.c_int32), _p(sh, C.c_double))
    if rc:
        raise ValueError("orc_estimate_shifts: %d" % rc)
    return SimpleNamespace(ishift=ish, shift=sh)


def footprint(w, h, sx, sy):
    fp = np.zeros(4, np.int32)
    lib().orc_footprint(C.c_int(w), C.c_int(h), C.c_double(sx), C.c_double(sy), _p(fp, C.c_int32))
    return fp


def resample(frames, sx, sy, fill=0.0, want64=False, interp=SPLINE):
    frames = _f32(frames)
    n, h, w = frames.shape
    sx = np.ascontiguousarray(np.broadcast_to(np.asarray(sx, np.float64), (n,)))
    sy = np.ascontiguousarray(np.broadcast_to(np.asarray(sy, np.float64), (n,)))
    out32 = np.empty((n, h, w), np.float32)
    out64 = np.empty((n, h, w), np.float64) if want64 else None
    fp = np.zeros((n, 4), np.int32)
    rc = lib().orc_resample_interp(_p(frames, C.c_float), C.c_int(n), C.c_int(w), C.c_int(h),
                                   _p(sx, C.c_double), _p(sy, C.c_double), C.c_double(fill), C.c_int(interp),
                                   _p(out64, C.c_double), _p(out32, C.c_float), _p(fp, C.c_int32))
    if rc:
        raise ValueError("orc_resample: %d" % rc)
    return SimpleNamespace(out=out32, out64=out64, footprint=fp)


def shift_line(f, s):
    f = np.ascontiguousarray(f, dtype=np.float64)
    out = np.empty_like(f)
    ok = np.zeros(f.shape[0], np.uint8)
    lib().orc_shift_line(_p(f, C.c_double), C.c_int(f.shape[0]), C.c_double(s), _p(out, C.c_double),
                         _p(ok, C.c_uint8))
    return out, ok.astype(bool)


def coadd(stack, footprint=None, mode=SIGCLIP, ksigma=3.0, max_iter=3, want64=False, want_mask=True):
    stack = _f32(stack)
    n, h, w = stack.shape
    if footprint is not None:
        footprint = np.ascontiguousarray(footprint, dtype=np.int32)
        assert footprint.shape == (n, 4)
    out32 = np.empty((h, w), np.float32)
    out64 = np.empty((h, w), np.float64) if want64 else None
    cnt = np.empty((h, w), np.uint16)
    words = (n + 31) // 32
    mask = np.empty((words, h, w), np.uint32) if want_mask else None
    margin = np.empty((h, w), np.float64)
    rc = lib().orc_coadd(_p(stack, C.c_float), C.c_int(n), C.c_int(w), C.c_int(h), _p(footprint, C.c_int32),
                         C.c_int(mode), C.c_double(ksigma), C.c_int(max_iter),
                         _p(out64, C.c_double), _p(out32, C.c_float), _p(cnt, C.c_uint16),
                         _p(mask, C.c_uint32), _p(margin, C.c_double))
    if rc:
        raise ValueError("orc_coadd: %d" % rc)
    return SimpleNamespace(out=out32, out64=out64, count=cnt, rejmask=mask, margin=margin)


def fill_bad(frames, badmask):
    """O7 (reading Q25): masked pixels replaced by linear interpolation along the short axis.  Returns a new array."""
    out = np.array(_f32(frames), copy=True)
    n, h, w = out.shape
    badmask = np.ascontiguousarray(badmask, dtype=np.uint8)
    assert badmask.shape == (h, w)
    rc = lib().orc_fill_bad(_p(out, C.c_float), C.c_int(n), C.c_int(w), C.c_int(h), _p(badmask, C.c_uint8))
    if rc:
        raise ValueError("orc_fill_bad: %d" % rc)
    return out
