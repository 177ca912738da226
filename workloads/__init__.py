"""Seeded synthetic BEST-2-shaped workloads (inputs only -- none of the method's arithmetic).

These stand in for the paper's simulated-pulsar benchmark file and BEST-2 recordings
(PAPER.md:190,194,214), neither of which is available.  Recipes: DESIGN.md section 4
(from BASELINE.json ``configs`` and SURVEY.md section 8(d)).  The same arrays are fed to
the CPU oracle and to the CUDA library; this module is imported by tests/ and bench.py
and imports neither of them.
"""
from .configs import CONFIGS, Config, generate, generate_beam, generate_beam_device, power_filterbank  # noqa: F401
