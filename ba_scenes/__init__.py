"""Seeded synthetic bundle-adjustment scenes (inputs only).

This module is the one piece shared by the fp64 oracle (`oracle/`) and the
CUDA path (`paper_2605_30583_b200/`).  It holds no solver arithmetic: it draws
cameras, points and visibility from a seeded `numpy` generator and synthesises
pixel measurements with scipy's rotation routine.  See DESIGN.md "Input recipe".
"""
from .generator import CONFIGS, FULL_OBSERVATIONS, Scene, make_scene, scene_summary  # noqa: F401
