"""Seeded synthetic inputs for the delta-checkpoint hot path.

This package serves BOTH the CPU oracle and the CUDA path and therefore holds none of
the method's arithmetic: no page compare, no CRC, no record layout.  It only makes
regions and mutates them, with the shapes of BASELINE.json's five configs
(recipes: DESIGN.md "Synthetic inputs").
"""
from .workloads import *  # noqa: F401,F403
