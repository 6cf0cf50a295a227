"""Oracle for the direct fine -> coarse summation of Eq. B.7.

ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).  Plain numpy, fp64.

PAPER.md:L454-L461 (Appendix B, Eq. B.7): instead of the quadrupled grid, the input of a fine grid s to the
potential on a coarser grid d is summed directly,

    Phi_ds^{s->d}(x_i, y_j, z_k) = -G sum_{i',j',k'} M^{m=s}(x_i', y_j', z_k') / |r_{ijk} - r_{i'j'k'}|,

M = rho dx_s^3 the cell masses of grid s, the distance taken between the CENTRE of the coarse cell and the
centres of the fine cells.  The grids are concentric (cell centre of index i on level l: (i + 1/2 - N/2) dx_l),
and for s > d a coarse centre is a corner of fine cells, so the distance never vanishes and no own-cell term
arises.  The paper finds this faster than the FFT route for N <= 32 (L461).
"""
from __future__ import annotations

import numpy as np


def direct_sum(rho_src: np.ndarray, dx0: float, src_level: int, dst_level: int, G: float = 1.0, targets=None) -> np.ndarray:
    """Phi_ds on every cell of level dst_level ([N,N,N]), or at the listed target cells [(k,j,i), ...]."""
    assert src_level > dst_level >= 0
    rho_src = np.asarray(rho_src, dtype=np.float64)
    N = rho_src.shape[0]
    dxs, dxd = dx0 / 2.0 ** src_level, dx0 / 2.0 ** dst_level
    cs = (np.arange(N) + 0.5 - N / 2) * dxs
    cd = (np.arange(N) + 0.5 - N / 2) * dxd
    Zs, Ys, Xs = np.meshgrid(cs, cs, cs, indexing="ij")
    M = (rho_src * dxs ** 3).ravel()
    Zs, Ys, Xs = Zs.ravel(), Ys.ravel(), Xs.ravel()
    cells = [(k, j, i) for k in range(N) for j in range(N) for i in range(N)] if targets is None else list(targets)
    out = np.empty(len(cells))
    for n, (k, j, i) in enumerate(cells):
        d = np.sqrt((cd[k] - Zs) ** 2 + (cd[j] - Ys) ** 2 + (cd[i] - Xs) ** 2)
        out[n] = -G * np.sum(M / d)
    return out.reshape(N, N, N) if targets is None else out
