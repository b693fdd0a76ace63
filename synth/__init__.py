"""Seeded synthetic inputs (scenes, cameras, trajectories) for the TemporalGS hot path.

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA path
(`paper_2607_03390_b200/`).  It holds none of the method's arithmetic: it only draws the
random Gaussians and the camera poses of the five workloads of `BASELINE.json:configs`
(recipe: DESIGN.md §4).  It imports neither `oracle` nor the CUDA package.
"""
from .scenes import Scene, Camera, make_config, CONFIG_NAMES, look_at  # noqa: F401
