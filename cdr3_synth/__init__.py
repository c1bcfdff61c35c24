"""Seeded synthetic CDR3-beta-shaped inputs (BASELINE.json `configs`).

This module is the ONLY code shared by the CPU oracle's tests and the CUDA
path's tests / bench.  It holds none of the method's arithmetic: no distance,
no threshold, no graph assembly — only random strings with the shapes the
paper's workloads have (SONIA-generated / empirical
CDR3-beta repertoires, which are not in this container; these inputs stand in
for them, recipe in DESIGN.md "Input recipe").
"""
from .generator import AA20, CONFIGS, SynthConfig, SynthData, generate, get_config

__all__ = ["AA20", "CONFIGS", "SynthConfig", "SynthData", "generate", "get_config"]
