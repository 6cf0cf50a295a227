"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic (no Green's function, no
restriction/prolongation, no FFT convolution): it only lays out the nested-grid
geometry the paper states (Fig. 1) and evaluates density
shapes on cell centres. It is the one module that both the oracle-side tests
and the CUDA-side tests/bench import, so both sides see the same arrays.
"""
from .configs import (CONFIGS, SEED0, cell_centres, dx_level, make_rho,
                      volume_fraction, level_rng)

__all__ = ["CONFIGS", "SEED0", "cell_centres", "dx_level", "make_rho",
           "volume_fraction", "level_rng"]
