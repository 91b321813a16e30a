"""Seeded synthetic input generators shared by the CPU oracle and the CUDA path.

This module holds NONE of the method's arithmetic (no transforms, no
contractions, no eigen-solves of chi): it only builds the *inputs* the C-ABI
takes -- cell, FFT grid, Miller-index spheres, v(q+G), plane-wave coefficients,
band energies and the frequency quadrature -- following the recipe of
BASELINE.json `configs` under the readings R1-R4, R11-R14 of SURVEY.md 8(c)
(restated in DESIGN.md "Input recipe").
"""
from .generate import (CONFIGS, RpaConfig, RpaInputs, make_inputs, sphere,
                       reciprocal_lattice, coulomb, quadrature, sweep_n_eig, SWEEP_FRACTIONS)

__all__ = ["CONFIGS", "RpaConfig", "RpaInputs", "make_inputs", "sphere",
           "reciprocal_lattice", "coulomb", "quadrature", "sweep_n_eig", "SWEEP_FRACTIONS"]
