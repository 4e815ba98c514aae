"""Timing sweeps of single entry points at sizes OUTSIDE bench.py's configurations.

    python -m paper_2008_11486_b200.sweep masters  [--frames 33,64,128] [--mode median|mean|clip] [--once]
    python -m paper_2008_11486_b200.sweep geometry
    python -m paper_2008_11486_b200.sweep coadd
    python -m paper_2008_11486_b200.sweep fill
    python -m paper_2008_11486_b200.sweep estimate

Every figure is the median of a few calls timed with CUDA events on the current stream, a 512 MB write between calls to
flush the L2.  Inputs are random numbers of the right type and range (timing only; parity is the business of tests/).
`--once` makes one warm call and one timed call and nothing else: the form to put under ncu
(profiles/r2_kernels.md names the commands).  The numbers these sweeps gave are in DESIGN.md section 7 and
profiles/r2_kernels.md.
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from . import binding as mred

PAPER = (1074, 1024, 0, 50, 50, 0, 1024, 1024)      # (W, H, os_x0, os_x1, x0, y0, w, h): PAPER.md L63
MODES = {"median": mred.MEDIAN, "mean": mred.MEAN, "clip": mred.SIGCLIP}
_flush = None


def _time_us(fn, reps=5, once=False):
    global _flush
    if _flush is None:
        _flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(1 if once else 2):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(1 if once else reps):
        _flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    return float(np.median(ts)) * 1e3


def _u16(n, g, lo, hi):
    return torch.randint(lo, hi, (n, g[1], g[0]), device="cuda", dtype=torch.int32).to(torch.uint16)


def masters(frames, modes, once):
    g = PAPER
    for n in frames:
        b, d, f = _u16(n, g, 400, 600), _u16(n, g, 400, 700), _u16(n, g, 15000, 25000)
        for nm in modes:
            us = _time_us(lambda: mred.build_masters(g, b, d, 60.0, f, 5.0, mode=MODES[nm]), once=once)
            print("build_masters 3 x %d frames %s: %.1f us (%.0f GB/s of input)" % (n, nm, us, 3 * b.numel() * 2 / us / 1e3), flush=True)


def geometry():
    n = 60
    geoms = {"paper": PAPER, "odd x0": (1077, 1024, 0, 53, 53, 0, 1024, 1024), "odd W": (1075, 1024, 0, 50, 50, 0, 1024, 1024),
             "w % 4 = 2": (1076, 1024, 0, 50, 50, 0, 1026, 1024), "w odd": (1073, 1024, 0, 50, 50, 0, 1023, 1024),
             "y0 = 3, h = 1000": (1074, 1024, 0, 50, 50, 3, 1024, 1000), "no overscan": (1024, 1024, 0, 0, 0, 0, 1024, 1024)}
    for nm, g in geoms.items():
        w, h = g[6], g[7]
        raw = _u16(n, g, 400, 3000)
        MB, MD, MF = torch.zeros((h, w), device="cuda"), torch.zeros((h, w), device="cuda"), torch.ones((h, w), device="cuda")
        out = torch.empty((n, h, w), device="cuda")
        us = _time_us(lambda: mred.calibrate(g, raw, 1.0, MB, MD, MF, out=out))
        print("%-17s calibrate %d frames: %.1f us" % (nm, n, us), flush=True)
        b = raw[:20].contiguous()
        us = _time_us(lambda: mred.build_masters(g, b, b, 60.0, b, 5.0, mode=mred.MEDIAN))
        print("%-17s build_masters 3 x 20: %.1f us" % (nm, us), flush=True)
        plan = mred.ReducePlan(g, n)
        us = _time_us(lambda: mred.reduce(plan, raw, 1.0, MB, MD, MF))
        print("%-17s reduce %d frames: %.1f us" % (nm, n, us), flush=True)


def coadd():
    h = w = 1024
    for n in (5, 10, 60):
        x = torch.randn((n, h, w), device="cuda") * 30 + 1000
        fp = np.tile(np.array([0, w - 1, 0, h - 1], np.int32), (n, 1))
        for nm, md in (("median", mred.MEDIAN), ("mean", mred.MEAN), ("clip", mred.SIGCLIP), ("minmax", mred.MINMAX), ("medclip", mred.MEDCLIP)):
            us = _time_us(lambda: mred.coadd(x, fp, mode=md))
            print("coadd %d x %d x %d %s: %.1f us" % (n, h, w, nm, us), flush=True)


def fill():
    n, h, w = 60, 1024, 1024
    x = torch.randn((n, h, w), device="cuda") * 30 + 1000
    rng = np.random.default_rng(3)
    masks = {}
    m = np.zeros((h, w), np.uint8); m[:, rng.choice(w, 10, replace=False)] = 1; masks["10 hot columns"] = m
    masks["5 % at random"] = (rng.random((h, w)) < 0.05).astype(np.uint8)
    m = np.zeros((h, w), np.uint8); m[400:500, 300:400] = 1; masks["100 x 100 blob"] = m
    m = np.zeros((h, w), np.uint8); m[100:110, :] = 1; masks["10 dead rows"] = m
    masks["50 % at random"] = (rng.random((h, w)) < 0.5).astype(np.uint8)
    m = np.ones((h, w), np.uint8); m[0, 0] = 0; masks["all but one pixel"] = m
    for nm, m in masks.items():
        md = torch.from_numpy(m).cuda()
        y = x.clone()
        us = _time_us(lambda: mred.fill_bad(y, md), reps=3)
        print("fill_bad %d frames, %s (%.2f %% masked): %.1f us" % (n, nm, 100 * m.mean(), us), flush=True)


def estimate():
    for (n, h, w) in ((60, 1024, 1024), (20, 4096, 4096), (255, 512, 512)):
        x = torch.randn((n, h, w), device="cuda") * 30 + 1000
        for lag in (8, 32, 64, 128, 255):
            us = _time_us(lambda: mred.estimate_shifts(x, 0, lag))
            print("estimate_shifts (stand-alone) %d x %d x %d, max_lag %d: %.1f us" % (n, h, w, lag, us), flush=True)
        del x


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("what", choices=["masters", "geometry", "coadd", "fill", "estimate"])
    ap.add_argument("--frames", default="10,20,32,33,48,64,80,96,100,128,130,192,255")
    ap.add_argument("--mode", default="median,mean,clip")
    ap.add_argument("--once", action="store_true")
    a = ap.parse_args()
    mred.lib()
    if a.what == "masters":
        masters([int(v) for v in a.frames.split(",")], a.mode.split(","), a.once)
    else:
        {"geometry": geometry, "coadd": coadd, "fill": fill, "estimate": estimate}[a.what]()


if __name__ == "__main__":
    main()
