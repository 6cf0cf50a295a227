"""Oracle for the modified ("dipole") convolution method over neighbouring pairs.

ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).  Written from the paper step
by step on top of the oracle's own primitives; shares nothing with the CUDA path.

PAPER.md:L282-L288 (Sect. 7, Fig. 14, Eq. 15) and L426-L433 (Appendix B, Eq. B.1-B.2): the original
method lets a coarse grid see the finer grid's mass only through its projection, which cancels dipole
(and higher) moments.  For every pair of neighbouring grids n : n+1 the fine grid is therefore expanded
to the physical size of the coarse one — a doubled grid Omega_dbl^{n+1} of (2N)^3 cells of the FINE size,
zero outside the original fine grid — its potential is found by the same convolution, reduced to the
coarse grid and added to the potential of the coarse grid with a cavity:

    Phi(Omega^n) = Phi_hole^{m=n} + tilde Phi_dbl^{m=n+1} + sum_{k<n} tilde Phi_hole^{m=k},   n < M_depth   (B.1)
    Phi(Omega^n) = Phi^{m=n} + sum_{k<n} tilde Phi_hole^{m=k},                                  n = M_depth   (B.2)

Readings: the density on the doubled grid is the fine grid's density as the original
method uses it (finer levels projected onto it, L280-L282); "reduced to the coarse grid" (the tilde
in the fine -> coarse direction, L288: unspecified) = arithmetic mean of the 8 fine-size cells that make
up a coarse cell (the same average as Eq. A.2); the coarse -> fine sum is the cascade of the original
method, unchanged.
"""
from __future__ import annotations

import numpy as np

from .cm_accel import child_mean
from .cm_oracle import field_direct, field_fft, green_hat, prolong, restrict


def doubled_density(rhobar_fine: np.ndarray) -> np.ndarray:
    """(2N)^3 array at the fine cell size, concentric with the fine grid: the fine grid's density in the
    central N^3 cells, zero in the added layers (Fig. 14)."""
    N = rhobar_fine.shape[0]
    out = np.zeros((2 * N, 2 * N, 2 * N))
    h = N // 2
    out[h:h + N, h:h + N, h:h + N] = rhobar_fine
    return out


def solve_modified(rho: np.ndarray, dx0: float, G: float = 1.0, method: str = "fft", return_parts: bool = False):
    """rho [L,N,N,N] -> Phi [L,N,N,N] by Eq. B.1-B.2 (pairs of neighbouring grids)."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    L, N = rho.shape[0], rho.shape[1]
    rhobar = restrict(rho)
    ghat = green_hat(N) if method == "fft" else None
    ghat2 = green_hat(2 * N) if (method == "fft" and L > 1) else None

    def field(a, hole, dx, gh):
        if method == "direct":
            return field_direct(a, hole, G, dx)
        return field_fft(a, hole, G, dx, gh)

    phi = np.empty_like(rho)
    ext = np.zeros((N, N, N))
    parts = {"dbl": [], "hole": [], "ext": []}
    for l in range(L):
        dx = dx0 / (1 << l)
        parts["ext"].append(ext)
        if l < L - 1:
            hole = field(rhobar[l], True, dx, ghat)
            dbl = field(doubled_density(rhobar[l + 1]), False, dx / 2.0, ghat2)   # on the doubled grid, fine cell size
            phi[l] = hole + child_mean(dbl) + ext                                  # B.1
            parts["hole"].append(hole)
            parts["dbl"].append(dbl)
            ext = prolong(ext + hole)
        else:
            phi[l] = field(rhobar[l], False, dx, ghat) + ext                       # B.2
    return (phi, parts) if return_parts else phi
