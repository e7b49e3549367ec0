"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds NONE of the method's arithmetic: it only draws truth-particle lists (pid, charge,
momentum, energy, vertex) with numpy's PCG64 and lays them out as CSR arrays.  The recipes are the ones
of BASELINE.json `configs[0..4]` as read in SURVEY.md section 8d / DESIGN.md "Input recipe"; they stand in
for the paper's Pythia8 samples, which are not available.
"""
from .generate import CONFIGS, Events, generate, config_card, concat_events, slice_events  # noqa: F401
