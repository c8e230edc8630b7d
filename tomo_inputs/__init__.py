"""Seeded synthetic workloads shared by the oracle tests and the CUDA-path tests.

This package holds *inputs only*: the five BASELINE.json configurations as plain
data (`configs.py`) and the von Karman phase-screen / slope generator
(`screens.py`).  It contains none of the reconstruction method's arithmetic
(no covariance, no Toeplitz/FFT product, no CG) and imports neither `oracle/`
nor `paper_1806_07938_b200/`.
"""
from .configs import TomoConfig, WFS, get_config, CONFIG_NAMES, sweep_config  # noqa: F401
