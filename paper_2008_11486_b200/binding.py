"""Thin ctypes binding of libmred.so (include/mred.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used for device
memory and streams.  There is no CPU fallback: a missing library or a non-zero status raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmred.so")

MEDIAN, MEAN, SIGCLIP, MINMAX, MEDCLIP = 0, 1, 2, 3, 4
PEAK_PARABOLA, PEAK_GAUSSIAN = 0, 1
INTERP_SPLINE, INTERP_BILINEAR, INTERP_NEAREST = 0, 1, 2
CALL_BUILD_MASTERS, CALL_CALIBRATE, CALL_ESTIMATE_SHIFTS, CALL_RESAMPLE, CALL_COADD, CALL_REDUCE, CALL_FILL_BAD = range(7)
MAX_STACK = 255

EXPORTS = ["mred_build_masters", "mred_calibrate", "mred_estimate_shifts", "mred_resample", "mred_coadd",
           "mred_reduce", "mred_reduce_staged", "mred_reduce_host", "mred_workspace_bytes", "mred_reduce_host_workspace_bytes",
           "mred_reduce_workspace_views", "mred_fill_bad", "mred_reduce_filled", "mred_estimate_shifts_peak", "mred_resample_interp",
           "mred_estimate_shifts_static", "mred_reduce_host_overlapped",
           "mred_strerror", "mred_last_cuda_error", "mred_version"]


class MredError(RuntimeError):
    pass


class Geom(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("W", "H", "os_x0", "os_x1", "x0", "y0", "w", "h")]


class CombOpts(C.Structure):
    _fields_ = [("mode", C.c_int32), ("ksigma", C.c_float), ("max_iter", C.c_int32)]


_lib = None


def lib():
    """Load libmred.so; raise loudly if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise MredError("libmred.so not found at %s: run `python -m paper_2008_11486_b200.build`" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        L.mred_strerror.restype = C.c_char_p
        L.mred_version.restype = C.c_char_p
        L.mred_workspace_bytes.restype = C.c_size_t
        L.mred_reduce_host_workspace_bytes.restype = C.c_size_t
        _lib = L
    return _lib


def _check(rc, what):
    if rc != 0:
        L = lib()
        msg = L.mred_strerror(C.c_int(rc)).decode()
        if rc == -4:
            msg += " (cudaError %d)" % L.mred_last_cuda_error()
        raise MredError("%s: %s" % (what, msg))


def geom(g) -> Geom:
    if isinstance(g, Geom):
        return g
    t = g.astuple() if hasattr(g, "astuple") else tuple(g)
    return Geom(*[int(v) for v in t])


def _dev(t, dtype, name):
    if t is None:
        return C.c_void_p(None)
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise MredError("%s must be a contiguous CUDA tensor of dtype %s" % (name, dtype))
    return C.c_void_p(t.data_ptr())


def _shape(t, shape, name):
    """Every tensor is checked against the geometry and frame count before the C ABI sees its pointer: the library
    trusts sizes, so a mismatched tensor would be read or written out of bounds."""
    if t is not None and tuple(t.shape) != tuple(shape):
        raise MredError("%s has shape %s, expected %s" % (name, tuple(t.shape), tuple(shape)))


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _opts(mode, ksigma, max_iter):
    return CombOpts(int(mode), float(ksigma), int(max_iter))


def workspace_bytes(call, g, n) -> int:
    gg = geom(g)
    return int(lib().mred_workspace_bytes(C.c_int(call), C.byref(gg), C.c_int(n)))


def reduce_host_workspace_bytes(g, n) -> int:
    gg = geom(g)
    return int(lib().mred_reduce_host_workspace_bytes(C.byref(gg), C.c_int(n)))


def _ws(ws, need, device):
    if ws is None:
        ws = torch.empty(max(need, 16), dtype=torch.uint8, device=device)
    return ws


def build_masters(g, bias, dark, t_dark, flat, t_flat, mode=MEDIAN, ksigma=3.0, max_iter=3, ws=None, stream=None,
                  out=None):
    """include/mred.h: mred_build_masters.  Returns (MB, MD, MF) float32 [h][w] CUDA tensors."""
    gg = geom(g)
    dev = bias.device
    MB, MD, MF = out if out is not None else [torch.empty((gg.h, gg.w), dtype=torch.float32, device=dev) for _ in range(3)]
    for t, nm in ((bias, "bias"), (dark, "dark"), (flat, "flat")):
        _shape(t, (t.shape[0], gg.H, gg.W), nm)
    for t, nm in ((MB, "MB"), (MD, "MD"), (MF, "MF")):
        _shape(t, (gg.h, gg.w), nm)
    nmax = max(bias.shape[0], dark.shape[0], flat.shape[0])
    ws = _ws(ws, workspace_bytes(CALL_BUILD_MASTERS, gg, nmax), dev)
    o = _opts(mode, ksigma, max_iter)
    rc = lib().mred_build_masters(C.byref(gg), _dev(bias, torch.uint16, "bias"), C.c_int(bias.shape[0]),
                                  _dev(dark, torch.uint16, "dark"), C.c_int(dark.shape[0]), C.c_float(t_dark),
                                  _dev(flat, torch.uint16, "flat"), C.c_int(flat.shape[0]), C.c_float(t_flat),
                                  C.byref(o), _dev(MB, torch.float32, "MB"), _dev(MD, torch.float32, "MD"),
                                  _dev(MF, torch.float32, "MF"), C.c_void_p(ws.data_ptr()), C.c_size_t(ws.numel()),
                                  _stream(stream))
    _check(rc, "mred_build_masters")
    return MB, MD, MF


def calibrate(g, raw, dark_scale, MB, MD, MF, out=None, level_out=None, ws=None, stream=None):
    """include/mred.h: mred_calibrate.  Returns (out float32 [n][h][w], level float64 [n])."""
    gg = geom(g)
    n = raw.shape[0]
    dev = raw.device
    if out is None:
        out = torch.empty((n, gg.h, gg.w), dtype=torch.float32, device=dev)
    if level_out is None:
        level_out = torch.empty(n, dtype=torch.float64, device=dev)
    _shape(raw, (n, gg.H, gg.W), "raw")
    for t, nm in ((MB, "MB"), (MD, "MD"), (MF, "MF")):
        _shape(t, (gg.h, gg.w), nm)
    _shape(out, (n, gg.h, gg.w), "out")
    _shape(level_out, (n,), "level_out")
    ws = _ws(ws, workspace_bytes(CALL_CALIBRATE, gg, n), dev)
    rc = lib().mred_calibrate(C.byref(gg), _dev(raw, torch.uint16, "raw"), C.c_int(n), C.c_float(dark_scale),
                              _dev(MB, torch.float32, "MB"), _dev(MD, torch.float32, "MD"),
                              _dev(MF, torch.float32, "MF"), _dev(out, torch.float32, "out"),
                              _dev(level_out, torch.float64, "level_out"), C.c_void_p(ws.data_ptr()),
                              C.c_size_t(ws.numel()), _stream(stream))
    _check(rc, "mred_calibrate")
    return out, level_out


def fill_bad(frames, badmask, ws=None, stream=None):
    """include/mred.h: mred_fill_bad.  In place on `frames` (float32 [n][h][w]); returns it."""
    n, h, w = frames.shape
    _shape(badmask, (h, w), "badmask")
    ws = _ws(ws, workspace_bytes(CALL_FILL_BAD, Geom(0, 0, 0, 0, 0, 0, w, h), n), frames.device)
    rc = lib().mred_fill_bad(_dev(frames, torch.float32, "frames"), C.c_int(n), C.c_int(w), C.c_int(h),
                             _dev(badmask, torch.uint8, "badmask"), C.c_void_p(ws.data_ptr()), C.c_size_t(ws.numel()),
                             _stream(stream))
    _check(rc, "mred_fill_bad")
    return frames


def estimate_shifts(frames, ref_index=0, max_lag=32, badmask=None, ws=None, stream=None, peak=0):
    """include/mred.h: mred_estimate_shifts.  Returns (ishift int32 [n][2], shift float64 [n][2]) on device."""
    n, h, w = frames.shape
    dev = frames.device
    ish = torch.empty((n, 2), dtype=torch.int32, device=dev)
    sh = torch.empty((n, 2), dtype=torch.float64, device=dev)
    _shape(badmask, (h, w), "badmask")
    gg = Geom(0, 0, 0, 0, 0, 0, w, h)
    ws = _ws(ws, workspace_bytes(CALL_ESTIMATE_SHIFTS, gg, n), dev)
    rc = lib().mred_estimate_shifts_peak(_dev(frames, torch.float32, "frames"), C.c_int(n), C.c_int(w), C.c_int(h),
                                         C.c_int(ref_index), C.c_int(max_lag), _dev(badmask, torch.uint8, "badmask"),
                                         C.c_int(peak), _dev(ish, torch.int32, "ishift"), _dev(sh, torch.float64, "shift"),
                                         C.c_void_p(ws.data_ptr()), C.c_size_t(ws.numel()), _stream(stream))
    _check(rc, "mred_estimate_shifts")
    return ish, sh


STATIC_SCRATCH_BYTES = 4 << 20


def estimate_shifts_static(frames, ishift, shift, ref_index=0, max_lag=32, badmask=None, stream=None, peak=0):
    """include/mred.h: mred_estimate_shifts_static -- no workspace and no allocation, here or in the library: the caller
    passes the outputs (ishift int32 [n][2], shift float64 [n][2], device).  MredError (MRED_ELIMIT) when the stack needs
    more than STATIC_SCRATCH_BYTES of scratch."""
    n, h, w = frames.shape
    _shape(badmask, (h, w), "badmask")
    _shape(ishift, (n, 2), "ishift")
    _shape(shift, (n, 2), "shift")
    rc = lib().mred_estimate_shifts_static(_dev(frames, torch.float32, "frames"), C.c_int(n), C.c_int(w), C.c_int(h),
                                           C.c_int(ref_index), C.c_int(max_lag), _dev(badmask, torch.uint8, "badmask"),
                                           C.c_int(peak), _dev(ishift, torch.int32, "ishift"),
                                           _dev(shift, torch.float64, "shift"), _stream(stream))
    _check(rc, "mred_estimate_shifts_static")
    return ishift, shift


def resample(frames, sx, sy, fill=0.0, out=None, ws=None, stream=None):
    """include/mred.h: mred_resample.  sx, sy: host float64 [n].  Returns (out, footprint int32 [n][4] numpy).
    ws: optional scratch of workspace_bytes(CALL_RESAMPLE, ...) bytes (allocated here when None and non-zero);
    ws=False passes no workspace, which selects the one-kernel route whatever the stack size."""
    n, h, w = frames.shape
    need = workspace_bytes(CALL_RESAMPLE, Geom(0, 0, 0, 0, 0, 0, w, h), n)
    if ws is False:
        ws = None
    elif ws is None and need:
        ws = torch.empty(need, dtype=torch.uint8, device=frames.device)
    sx = np.ascontiguousarray(np.broadcast_to(np.asarray(sx, np.float64), (n,)))
    sy = np.ascontiguousarray(np.broadcast_to(np.asarray(sy, np.float64), (n,)))
    if out is None:
        out = torch.empty_like(frames)
    _shape(out, (n, h, w), "out")
    fp = np.zeros((n, 4), np.int32)
    rc = lib().mred_resample(_dev(frames, torch.float32, "frames"), C.c_int(n), C.c_int(w), C.c_int(h),
                             sx.ctypes.data_as(C.c_void_p), sy.ctypes.data_as(C.c_void_p), C.c_float(fill),
                             _dev(out, torch.float32, "out"), fp.ctypes.data_as(C.c_void_p),
                             C.c_void_p(ws.data_ptr() if ws is not None else None),
                             C.c_size_t(ws.numel() if ws is not None else 0), _stream(stream))
    _check(rc, "mred_resample")
    return out, fp


def resample_interp(frames, sx, sy, interp, fill=0.0, out=None, stream=None):
    """include/mred.h: mred_resample_interp (bilinear / nearest / spline).  Returns (out, footprint int32 [n][4] numpy)."""
    n, h, w = frames.shape
    sx = np.ascontiguousarray(np.broadcast_to(np.asarray(sx, np.float64), (n,)))
    sy = np.ascontiguousarray(np.broadcast_to(np.asarray(sy, np.float64), (n,)))
    if out is None:
        out = torch.empty_like(frames)
    _shape(out, (n, h, w), "out")
    fp = np.zeros((n, 4), np.int32)
    rc = lib().mred_resample_interp(_dev(frames, torch.float32, "frames"), C.c_int(n), C.c_int(w), C.c_int(h),
                                    sx.ctypes.data_as(C.c_void_p), sy.ctypes.data_as(C.c_void_p), C.c_float(fill),
                                    C.c_int(interp), _dev(out, torch.float32, "out"), fp.ctypes.data_as(C.c_void_p),
                                    _stream(stream))
    _check(rc, "mred_resample_interp")
    return out, fp


def coadd(stack, footprint=None, mode=SIGCLIP, ksigma=3.0, max_iter=3, want_count=True, want_mask=False, stream=None):
    """include/mred.h: mred_coadd.  footprint: host int32 [n][4] or None.  Returns (out, count, rejmask)."""
    n, h, w = stack.shape
    dev = stack.device
    out = torch.empty((h, w), dtype=torch.float32, device=dev)
    count = torch.empty((h, w), dtype=torch.uint16, device=dev) if want_count else None
    mask = torch.empty(((n + 31) // 32, h, w), dtype=torch.uint32, device=dev) if want_mask else None
    fpp = C.c_void_p(None)
    if footprint is not None:
        footprint = np.ascontiguousarray(footprint, dtype=np.int32)
        if footprint.shape != (n, 4):
            raise MredError("footprint must be [n][4]")
        fpp = footprint.ctypes.data_as(C.c_void_p)
    o = _opts(mode, ksigma, max_iter)
    rc = lib().mred_coadd(_dev(stack, torch.float32, "stack"), C.c_int(n), C.c_int(w), C.c_int(h), fpp, C.byref(o),
                          _dev(out, torch.float32, "out"), _dev(count, torch.uint16, "count"),
                          _dev(mask, torch.uint32, "rejmask"), _stream(stream))
    _check(rc, "mred_coadd")
    return out, count, mask


class ReducePlan:
    """Pre-allocated buffers for mred_reduce / mred_reduce_host on one group shape (n frames)."""

    def __init__(self, g, n, device="cuda", want_count=True, want_mask=False, host=False):
        self.g = geom(g)
        self.n = n
        self.host = host
        dev = torch.device(device)
        need = reduce_host_workspace_bytes(self.g, n) if host else workspace_bytes(CALL_REDUCE, self.g, n)
        self.ws = torch.empty(need, dtype=torch.uint8, device=dev)
        h, w = self.g.h, self.g.w
        if host:
            self.out = torch.empty((h, w), dtype=torch.float32).pin_memory()
            self.count = torch.empty((h, w), dtype=torch.uint16).pin_memory() if want_count else None
            self.shift = torch.empty((n, 2), dtype=torch.float64).pin_memory()
            self.mask = None
            self.footprint = None
        else:
            self.out = torch.empty((h, w), dtype=torch.float32, device=dev)
            self.count = torch.empty((h, w), dtype=torch.uint16, device=dev) if want_count else None
            self.mask = torch.empty(((n + 31) // 32, h, w), dtype=torch.uint32, device=dev) if want_mask else None
            self.shift = torch.empty((n, 2), dtype=torch.float64, device=dev)
            self.footprint = torch.empty((n, 4), dtype=torch.int32, device=dev)

    def _view(self, which):
        """float32 [n][h][w] view of the calibrated (0) / registered (1) stack mred_reduce left in the workspace
        (mred_reduce_workspace_views); device plans only, valid until the plan is used again."""
        if self.host:
            raise MredError("workspace views exist for device plans only")
        offs = (C.c_size_t(0), C.c_size_t(0))
        _check(lib().mred_reduce_workspace_views(C.byref(self.g), C.c_int(self.n), C.byref(offs[0]), C.byref(offs[1])),
               "mred_reduce_workspace_views")
        nbytes = 4 * self.n * self.g.h * self.g.w
        o = offs[which].value
        return self.ws[o:o + nbytes].view(torch.float32).view(self.n, self.g.h, self.g.w)

    def calibrated(self):
        return self._view(0)

    def registered(self):
        return self._view(1)


def _reduce_shapes(plan, raw, MB, MD, MF, badmask):
    g = plan.g
    _shape(raw, (plan.n, g.H, g.W), "raw")
    for t, nm in ((MB, "MB"), (MD, "MD"), (MF, "MF"), (badmask, "badmask")):
        _shape(t, (g.h, g.w), nm)


def reduce(plan: ReducePlan, raw, dark_scale, MB, MD, MF, ref_index=0, max_lag=32, badmask=None, fill=0.0,
           mode=SIGCLIP, ksigma=3.0, max_iter=3, stream=None, events=None, fill_bad=False):
    """include/mred.h: mred_reduce / mred_reduce_staged (device-resident chained science path).  Results land
    in `plan`.  events: optional list of 5 torch.cuda.Event(enable_timing=True) recorded around the stages."""
    _reduce_shapes(plan, raw, MB, MD, MF, badmask)
    o = _opts(mode, ksigma, max_iter)
    if fill_bad:       # include/mred.h: mred_reduce_filled (no stage events)
        if badmask is None or events is not None:
            raise MredError("fill_bad needs a badmask and takes no stage events")
        rc = lib().mred_reduce_filled(C.byref(plan.g), _dev(raw, torch.uint16, "raw"), C.c_int(plan.n), C.c_float(dark_scale),
                           _dev(MB, torch.float32, "MB"), _dev(MD, torch.float32, "MD"), _dev(MF, torch.float32, "MF"),
                           C.c_int(ref_index), C.c_int(max_lag), _dev(badmask, torch.uint8, "badmask"),
                           C.c_float(fill), C.byref(o), _dev(plan.out, torch.float32, "out"),
                           _dev(plan.count, torch.uint16, "count"), _dev(plan.mask, torch.uint32, "rejmask"),
                           _dev(plan.shift, torch.float64, "shift"), _dev(plan.footprint, torch.int32, "footprint"),
                           C.c_void_p(plan.ws.data_ptr()), C.c_size_t(plan.ws.numel()), _stream(stream))
        _check(rc, "mred_reduce_filled")
        return plan
    ev = C.c_void_p(None)
    if events is not None:
        for e in events:
            if e.cuda_event == 0:      # torch creates the CUDA event lazily, on first record
                e.record(torch.cuda.current_stream() if stream is None else stream)
        ev = (C.c_void_p * 5)(*[C.c_void_p(e.cuda_event) for e in events])
    rc = lib().mred_reduce_staged(C.byref(plan.g), _dev(raw, torch.uint16, "raw"), C.c_int(plan.n), C.c_float(dark_scale),
                           _dev(MB, torch.float32, "MB"), _dev(MD, torch.float32, "MD"), _dev(MF, torch.float32, "MF"),
                           C.c_int(ref_index), C.c_int(max_lag), _dev(badmask, torch.uint8, "badmask"),
                           C.c_float(fill), C.byref(o), _dev(plan.out, torch.float32, "out"),
                           _dev(plan.count, torch.uint16, "count"), _dev(plan.mask, torch.uint32, "rejmask"),
                           _dev(plan.shift, torch.float64, "shift"), _dev(plan.footprint, torch.int32, "footprint"),
                           C.c_void_p(plan.ws.data_ptr()), C.c_size_t(plan.ws.numel()), _stream(stream), ev)
    _check(rc, "mred_reduce")
    return plan


def reduce_host(plan: ReducePlan, raw_host, dark_scale, MB, MD, MF, ref_index=0, max_lag=32, badmask=None, fill=0.0,
                mode=SIGCLIP, ksigma=3.0, max_iter=3, stream=None):
    """include/mred.h: mred_reduce_host.  raw_host: CPU (pinned) uint16 tensor [n][H][W]; the co-add, count
    and shifts come back in plan.out / plan.count / plan.shift (pinned host tensors)."""
    if raw_host.is_cuda or raw_host.dtype != torch.uint16 or not raw_host.is_contiguous():
        raise MredError("raw_host must be a contiguous CPU uint16 tensor")
    if not plan.host:
        raise MredError("reduce_host needs a ReducePlan(host=True)")
    _reduce_shapes(plan, raw_host, MB, MD, MF, badmask)
    o = _opts(mode, ksigma, max_iter)
    rc = lib().mred_reduce_host(C.byref(plan.g), C.c_void_p(raw_host.data_ptr()), C.c_int(plan.n),
                                C.c_float(dark_scale), _dev(MB, torch.float32, "MB"), _dev(MD, torch.float32, "MD"),
                                _dev(MF, torch.float32, "MF"), C.c_int(ref_index), C.c_int(max_lag),
                                _dev(badmask, torch.uint8, "badmask"), C.c_float(fill), C.byref(o),
                                C.c_void_p(plan.out.data_ptr()),
                                C.c_void_p(plan.count.data_ptr() if plan.count is not None else None),
                                C.c_void_p(plan.shift.data_ptr()), C.c_void_p(plan.ws.data_ptr()),
                                C.c_size_t(plan.ws.numel()), _stream(stream))
    _check(rc, "mred_reduce_host")
    return plan


HOST_CHUNKS = 4


def reduce_host_overlapped(plan: ReducePlan, raw_host, dark_scale, MB, MD, MF, copy_stream, events, ref_index=0, max_lag=32,
                           badmask=None, fill=0.0, mode=SIGCLIP, ksigma=3.0, max_iter=3, stream=None):
    """include/mred.h: mred_reduce_host_overlapped -- mred_reduce_host with the host->device copy in HOST_CHUNKS pieces on
    `copy_stream` (a torch.cuda.Stream other than `stream`), each piece calibrated while the next is on the bus.
    events: HOST_CHUNKS + 1 torch.cuda.Event objects, reusable from call to call.  Results as reduce_host."""
    if raw_host.is_cuda or raw_host.dtype != torch.uint16 or not raw_host.is_contiguous():
        raise MredError("raw_host must be a contiguous CPU uint16 tensor")
    if not plan.host:
        raise MredError("reduce_host_overlapped needs a ReducePlan(host=True)")
    if len(events) != HOST_CHUNKS + 1:
        raise MredError("events must hold HOST_CHUNKS + 1 torch.cuda.Event objects")
    _reduce_shapes(plan, raw_host, MB, MD, MF, badmask)
    o = _opts(mode, ksigma, max_iter)
    for e in events:
        if e.cuda_event == 0:          # torch creates the CUDA event lazily, on first record
            e.record(copy_stream)
    ev = (C.c_void_p * (HOST_CHUNKS + 1))(*[C.c_void_p(e.cuda_event) for e in events])
    rc = lib().mred_reduce_host_overlapped(C.byref(plan.g), C.c_void_p(raw_host.data_ptr()), C.c_int(plan.n),
                                           C.c_float(dark_scale), _dev(MB, torch.float32, "MB"), _dev(MD, torch.float32, "MD"),
                                           _dev(MF, torch.float32, "MF"), C.c_int(ref_index), C.c_int(max_lag),
                                           _dev(badmask, torch.uint8, "badmask"), C.c_float(fill), C.byref(o),
                                           C.c_void_p(plan.out.data_ptr()),
                                           C.c_void_p(plan.count.data_ptr() if plan.count is not None else None),
                                           C.c_void_p(plan.shift.data_ptr()), C.c_void_p(plan.ws.data_ptr()),
                                           C.c_size_t(plan.ws.numel()), _stream(stream), C.c_void_p(copy_stream.cuda_stream), ev)
    _check(rc, "mred_reduce_host_overlapped")
    return plan
