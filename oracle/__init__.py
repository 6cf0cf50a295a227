"""ORACLE — test infrastructure, not the product.

Plain CPU statement of the nested-grid convolution method of arXiv 2301.06763
(§3-§4, Eq. 10, 13, 14).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package; the
product (paper_2301_06763_b200) never does, and this package never imports the
product.
"""
from .cm_oracle import (build, lib, I0, restrict, field_direct, field_fft, green_hat,
                        prolong, solve, solve_points, leaf_direct, num_threads,
                        fft1d, dft_naive, field_direct_at)

from .cm_accel import acceleration, ghost_value, child_mean, padded_level
from .cm_modified import solve_modified, doubled_density, solve_modified_triplets, expanded_density, block_mean
from .cm_direct import direct_sum

__all__ = ["acceleration", "ghost_value", "child_mean", "padded_level", "solve_modified", "doubled_density", "solve_modified_triplets", "expanded_density", "block_mean", "direct_sum",
           "build", "lib", "I0", "restrict", "field_direct", "field_fft", "green_hat",
           "prolong", "solve", "solve_points", "leaf_direct", "num_threads",
           "fft1d", "dft_naive", "field_direct_at"]
