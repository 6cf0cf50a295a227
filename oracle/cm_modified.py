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


def expanded_density(rhobar_fine: np.ndarray, factor: int, hole: bool = False) -> np.ndarray:
    """(factor N)^3 array at the fine cell size, concentric with the fine grid: the fine grid's density in the
    central N^3 cells (with its own cavity [N/4, 3N/4)^3 zeroed if `hole`: the doubled grid "with a central hole"
    of the triplet scheme, L448), zero in the added layers.  factor 2 = Omega_dbl, 4 = Omega_qdp (Fig. B.1)."""
    N = rhobar_fine.shape[0]
    core = np.array(rhobar_fine, dtype=np.float64, copy=True)
    if hole:
        q = N // 4
        core[q:3 * q, q:3 * q, q:3 * q] = 0.0
    out = np.zeros((factor * N,) * 3)
    h = (factor - 1) * N // 2
    out[h:h + N, h:h + N, h:h + N] = core
    return out


def block_mean(a: np.ndarray, factor: int) -> np.ndarray:
    """Arithmetic mean over the factor^3 fine-size cells that make up each coarse cell (reading M2)."""
    n = a.shape[0] // factor
    return a.reshape(n, factor, n, factor, n, factor).mean(axis=(1, 3, 5))


def solve_modified_triplets(rho: np.ndarray, dx0: float, G: float = 1.0, qdp: str = "fft"):
    """rho [L,N,N,N] -> Phi [L,N,N,N] by Eq. B.3-B.6 (dipole moments across three neighbouring grids):

        Phi(Omega^n) = Phi_hole^n + tilde Phi_dbl,hole^{n+1} + tilde Phi_qdp^{n+2} + sum_{k<n} tilde Phi_hole^k   (B.3, n < M-1)
        Phi(Omega^n) = Phi_hole^n + tilde Phi_dbl^{n+1} + sum_{k<n} tilde Phi_hole^k                            (B.5, n = M-1)
        Phi(Omega^n) = Phi^n + sum_{k<n} tilde Phi_hole^k                                                       (B.6, n = M)

    qdp = "fft": the quadrupled grid (4N)^3 of Fig. B.1 by the same convolution, reduced by the mean over the 4^3
    fine-size cells of a coarse cell; qdp = "direct": Eq. B.7 instead (cm_direct.direct_sum)."""
    from .cm_direct import direct_sum
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    L, N = rho.shape[0], rho.shape[1]
    rhobar = restrict(rho)
    gh = {1: green_hat(N)}
    phi = np.empty_like(rho)
    ext = np.zeros((N, N, N))
    for l in range(L):
        dx = dx0 / (1 << l)
        if l == L - 1:
            phi[l] = field_fft(rhobar[l], False, G, dx, gh[1]) + ext                                    # B.6
            continue
        hole = field_fft(rhobar[l], True, G, dx, gh[1])
        gh.setdefault(2, green_hat(2 * N))
        triple = l < L - 2
        dbl = field_fft(expanded_density(rhobar[l + 1], 2, hole=triple), False, G, dx / 2, gh[2])
        phi[l] = hole + block_mean(dbl, 2) + ext                                                        # B.5 / first terms of B.3
        if triple:
            if qdp == "fft":
                gh.setdefault(4, green_hat(4 * N))
                q = field_fft(expanded_density(rhobar[l + 2], 4), False, G, dx / 4, gh[4])
                phi[l] = phi[l] + block_mean(q, 4)
            else:
                phi[l] = phi[l] + direct_sum(rhobar[l + 2], dx0, l + 2, l, G=G)                         # B.7
        ext = prolong(ext + hole)
    return phi


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
