"""Seeded synthetic MITSuME-like CCD frames (input generator only).

This package holds NO arithmetic of the reduction method: it only draws the
detector-model inputs (raw uint16 frames, exposure times, true shifts, bad-pixel
mask) that both the CUDA path and the CPU oracle are fed.  Neither of those
imports the other; both may import this.
"""
from .frames import (Geom, CONFIGS, GEOM_MITSUME, GEOM_PAPER, GEOM_LARGE, GEOM_SMALL,  # noqa: F401
                     make_group, group_spec, bspline_bump_image, beta3,
                     MEDIAN, MEAN, SIGCLIP)
