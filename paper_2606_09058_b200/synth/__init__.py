"""Seeded synthetic NAO-shaped inputs (BASELINE.json configs 0-4).

This package is the ONE piece shared by the CPU oracle and the CUDA path: it only
generates inputs and holds none of the method's arithmetic.  See nao_synth.c and
DESIGN.md ("Input recipe").
"""
from .synth import CONFIGS, Problem, make_config, build_synth_lib, as_matrix  # noqa: F401
