"""Seeded synthetic CCD frames shaped like the paper's MITSuME data.

Stands in for the MITSuME-Akeno frames of 2018-05-14 / 2018-08-22 and the random
N x N dummy sets the paper measures on, none of which
exist here.  Recipe: SURVEY.md section 8(d) / DESIGN.md "Input recipe".

Detector model, per raw pixel (gain 1 e-/ADU):
    raw = clip(round(Poisson(flat(x,y) * [sky_k + sum(stars)] + 0.05 * t) + 500 + N(0, rn)), 0, 65535)
    overscan columns = round(500 + N(0, rn))
Nothing in this file belongs to the reduction method itself.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from types import SimpleNamespace

import numpy as np

BASE_SEED = 20200826          # the paper's acceptance date; seed = BASE + 1000*config + group
PEDESTAL = 500.0              # ADU
DARK_RATE = 0.05              # ADU / s
FLAT_LEVEL = 20000.0          # ADU of illumination in flat frames
T_DARK, T_FLAT, T_SCI = 60.0, 5.0, 60.0
STAR_SIGMA = 3.0 / 2.3548200450309493   # FWHM 3 px


@dataclass(frozen=True)
class Geom:
    """Raw-frame geometry: W x H raw (x fastest), overscan columns [os_x0, os_x1),
    image rectangle (x0, y0, w, h).  PAPER.md L49 (1074x1024 incl. overscan), L63."""
    W: int
    H: int
    os_x0: int
    os_x1: int
    x0: int
    y0: int
    w: int
    h: int

    def astuple(self):
        return (self.W, self.H, self.os_x0, self.os_x1, self.x0, self.y0, self.w, self.h)


GEOM_MITSUME = Geom(1074, 1024, 0, 50, 50, 0, 1024, 1024)     # BASELINE.json configs 1-4
GEOM_PAPER = Geom(1074, 1024, 0, 50, 52, 2, 1020, 1020)       # 1020 x 1020 after trim
GEOM_LARGE = Geom(4128, 4096, 0, 32, 32, 0, 4096, 4096)       # BASELINE.json config 5
GEOM_SMALL = Geom(210, 136, 0, 18, 18, 0, 192, 136)           # test-size stand-in, same structure

# combine modes (values match include/mred.h and oracle/mred_oracle.c by convention only)
MEDIAN, MEAN, SIGCLIP = 0, 1, 2

CONFIGS = {
    1: dict(geom=GEOM_MITSUME, groups=1, n_sci=5, n_master=3, stars=50, S=10.0, sky=(1000.0, 1000.0),
            rn=10.0, coadd=MEDIAN, stress=False),
    2: dict(geom=GEOM_MITSUME, groups=3, n_sci=10, n_master=10, stars=200, S=20.0, sky=(1000.0, 1000.0),
            rn=10.0, coadd=SIGCLIP, stress=False),
    3: dict(geom=GEOM_MITSUME, groups=6, n_sci=60, n_master=20, stars=300, S=30.0, sky=(500.0, 3000.0),
            rn=10.0, coadd=SIGCLIP, stress=False),
    4: dict(geom=GEOM_MITSUME, groups=1, n_sci=64, n_master=10, stars=200, S=10.0, sky=(1000.0, 1000.0),
            rn=10.0, coadd=SIGCLIP, stress=True),
    5: dict(geom=GEOM_LARGE, groups=1, n_sci=100, n_master=10, stars=1000, S=50.0, sky=(800.0, 800.0),
            rn=8.0, coadd=SIGCLIP, stress=False),
}


def group_spec(config: int, **over) -> dict:
    spec = dict(CONFIGS[config])
    spec.update({k: v for k, v in over.items() if v is not None})
    return spec


def _rng(seed, *path):
    return np.random.default_rng(np.random.SeedSequence([int(seed), *[int(p) for p in path]]))


def _flat_field(g: Geom):
    X = np.arange(g.W, dtype=np.float64) - g.x0
    Y = np.arange(g.H, dtype=np.float64) - g.y0
    fx = 2.0 * X / max(g.w - 1, 1) - 1.0
    fy = 2.0 * Y / max(g.h - 1, 1) - 1.0
    return 1.0 + 0.05 * (fx[None, :] + fy[:, None]) / 2.0


def _finish(rng, g: Geom, electrons, rn):
    """Poisson + pedestal + read noise, overscan columns bias-only, uint16."""
    img = rng.poisson(np.maximum(electrons, 0.0)).astype(np.float64)
    img += PEDESTAL + rng.normal(0.0, rn, size=img.shape)
    if g.os_x1 > g.os_x0:
        img[:, g.os_x0:g.os_x1] = PEDESTAL + rng.normal(0.0, rn, size=(g.H, g.os_x1 - g.os_x0))
    return np.clip(np.rint(img), 0, 65535).astype(np.uint16)


def _render_stars(g: Geom, xs, ys, peaks):
    """Point-sampled Gaussians (FWHM 3 px) at image coordinates (xs, ys), on the raw grid."""
    sky = np.zeros((g.H, g.W), dtype=np.float64)
    r = 8
    for x, y, p in zip(xs, ys, peaks):
        X, Y = x + g.x0, y + g.y0
        ix, iy = int(np.floor(X)), int(np.floor(Y))
        xa, xb = max(ix - r, 0), min(ix + r + 1, g.W)
        ya, yb = max(iy - r, 0), min(iy + r + 1, g.H)
        if xa >= xb or ya >= yb:
            continue
        gx = np.exp(-0.5 * ((np.arange(xa, xb) - X) / STAR_SIGMA) ** 2)
        gy = np.exp(-0.5 * ((np.arange(ya, yb) - Y) / STAR_SIGMA) ** 2)
        sky[ya:yb, xa:xb] += p * gy[:, None] * gx[None, :]
    return sky


def _draw_shifts(rng, n, S):
    """True content displacement (dx, dy) of frame k w.r.t. frame 0; fractional part kept
    >= 0.05 away from +-0.5 so the nearest-integer estimate is not on its own tie."""
    sh = np.zeros((n, 2), dtype=np.float64)
    for k in range(1, n):
        for a in range(2):
            while True:
                v = rng.uniform(-S, S)
                fr = v - np.rint(v)
                if abs(abs(fr) - 0.5) >= 0.05 and abs(v) <= S:
                    break
            sh[k, a] = v
    return sh


def _map(fn, items, workers):
    """Frames are drawn from independent generators (one SeedSequence path each), so they can be made in any order
    and on several threads (numpy releases the GIL while it draws) with the same result."""
    items = list(items)
    if workers and workers > 1 and len(items) > 1:
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=min(workers, len(items))) as ex:
            return list(ex.map(fn, items))
    return [fn(i) for i in items]


def make_group(config: int, group: int = 0, *, geom: Geom | None = None, n_sci=None, n_master=None,
               stars=None, S=None, seed=None, masters: bool = True, science: bool = True, workers: int = 0):
    """One (telescope, band) group of BASELINE.json config `config`.

    Returns a namespace with uint16 stacks bias/dark/flat/sci of shape [n][H][W], exposure
    times, the true shifts (n_sci, 2), the co-add mode and, for the stress config, `badmask`
    (uint8 [h][w], 1 = hot column) -- otherwise None.  `geom`, counts, `stars`, `S` override
    the config for test-sized cases; the value model is unchanged.
    """
    sp = group_spec(config, geom=geom, n_sci=n_sci, n_master=n_master, stars=stars, S=S)
    g: Geom = sp["geom"]
    seed = BASE_SEED + 1000 * config + group if seed is None else seed
    rn = sp["rn"]
    flat = _flat_field(g)
    out = SimpleNamespace(config=config, group=group, geom=g, seed=seed, t_dark=T_DARK, t_flat=T_FLAT,
                          t_sci=T_SCI, coadd=sp["coadd"], ksigma=3.0, max_iter=3, S=sp["S"],
                          bias=None, dark=None, flat=None, sci=None, shifts=None, badmask=None, sky=None)
    nm = sp["n_master"]
    if masters:
        out.bias = np.stack(_map(lambda k: _finish(_rng(seed, 1, k), g, np.zeros((g.H, g.W)), rn), range(nm), workers))
        out.dark = np.stack(_map(lambda k: _finish(_rng(seed, 2, k), g, np.full((g.H, g.W), DARK_RATE * T_DARK), rn),
                                 range(nm), workers))
        out.flat = np.stack(_map(lambda k: _finish(_rng(seed, 3, k), g, flat * FLAT_LEVEL + DARK_RATE * T_FLAT, rn),
                                 range(nm), workers))
    if not science:
        return out
    n = sp["n_sci"]
    r0 = _rng(seed, 4)
    S = sp["S"]
    ns = sp["stars"]
    sx = r0.uniform(-S, g.w + S, size=ns)
    sy = r0.uniform(-S, g.h + S, size=ns)
    peaks = np.exp(r0.uniform(np.log(200.0), np.log(20000.0), size=ns))
    if sp["stress"]:
        sat = r0.random(ns) < 0.05                      # 5 % of stars above saturation
        peaks = np.where(sat, r0.uniform(1.0e5, 3.0e5, size=ns), peaks)
    shifts = _draw_shifts(r0, n, S)
    skies = r0.uniform(sp["sky"][0], sp["sky"][1], size=n)
    hot_cols = hot_amp = None
    if sp["stress"]:
        nh = max(1, int(round(0.01 * g.w)))             # "1 % hot columns"
        hot_cols = np.sort(r0.choice(g.w, size=nh, replace=False))
        hot_amp = r0.uniform(2000.0, 20000.0, size=nh)
        out.badmask = np.zeros((g.h, g.w), dtype=np.uint8)
        out.badmask[:, hot_cols] = 1
    def one_frame(k):
        rk = _rng(seed, 5, k)
        model = skies[k] + _render_stars(g, sx + shifts[k, 0], sy + shifts[k, 1], peaks)
        el = flat * model + DARK_RATE * T_SCI
        if hot_cols is not None:
            el[:, hot_cols + g.x0] += hot_amp[None, :]
        if sp["stress"]:                                 # cosmic rays: 1e-4 of pixels, 1-4 px tracks
            nhit = int(round(1.0e-4 * g.w * g.h))
            cx = rk.integers(0, g.w, size=nhit) + g.x0
            cy = rk.integers(0, g.h, size=nhit) + g.y0
            ln = rk.integers(1, 5, size=nhit)
            horiz = rk.random(nhit) < 0.5
            amp = rk.uniform(5000.0, 60000.0, size=nhit)
            for j in range(nhit):
                for s in range(ln[j]):
                    X = cx[j] + (s if horiz[j] else 0)
                    Y = cy[j] + (0 if horiz[j] else s)
                    if X < g.W and Y < g.H:
                        el[Y, X] += amp[j]
        return _finish(rk, g, el, rn)

    out.sci = np.stack(_map(one_frame, range(n), workers))
    out.shifts = shifts
    out.sky = skies
    return out


# ---------------------------------------------------------------------------------------------
# The paper's analytic test image (Fig. 8/9): cubic B-spline basis functions
# arranged on a grid.  A shifted copy is obtained "without actually interpolating".
# ---------------------------------------------------------------------------------------------
def beta3(t):
    """Cubic B-spline basis function (support [-2, 2], peak 2/3)."""
    a = np.abs(np.asarray(t, dtype=np.float64))
    return np.where(a < 1.0, 2.0 / 3.0 - a * a + 0.5 * a ** 3,
                    np.where(a < 2.0, (2.0 - a) ** 3 / 6.0, 0.0))


def bspline_bump_image(w, h, centres, p, amp=2000.0, sx=0.0, sy=0.0):
    """sum_m amp * beta3((x - sx - xm)/p) * beta3((y - sy - ym)/p) on the integer grid, float64.
    With integer p, xm, ym and supports clear of the edges this is a natural cubic spline with
    integer knots, so its translate by (sx, sy) is what an exact spline shift must return."""
    x = np.arange(w, dtype=np.float64) - sx
    y = np.arange(h, dtype=np.float64) - sy
    img = np.zeros((h, w), dtype=np.float64)
    for (xm, ym) in centres:
        img += amp * beta3((y - ym) / p)[:, None] * beta3((x - xm) / p)[None, :]
    return img
