"""Seeded synthetic input generator shared by the CUDA path and the oracle.

Holds NONE of the method's arithmetic: it draws parameter vectors from the priors
BASELINE.json lists, builds the static inputs (grids, PSFs, bin maps, MGE tables,
quadrature nodes) and adds noise to a noise-free truth model that the CALLER
supplies through `data_model` (tests pass the oracle, bench.py's GPU leg passes
the CUDA library).  Recipe and every reading: DESIGN.md "Input recipe".

These inputs stand in for the paper's simulated RXJ1131 HST-ACS image and
NIRSpec-like kinematic map (section 4), which are not
available; shapes/distributions follow BASELINE.json:configs first.
"""
from .generate import CONFIGS, make_workload, gauss_legendre_u, quasar_data, subset, pixsrc_inputs, kronrod_composite, jam_sph_rules, cse_table, enfw_params  # noqa: F401
