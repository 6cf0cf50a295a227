"""Oracle for the gravitational acceleration on the nested mesh.

ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).  Plain numpy,
fp64, written from the paper step by step; shares nothing with the CUDA path.

What it computes, level by level (PAPER.md line numbers):

  g = -grad Phi by the six-point central stencil                      (Eq. 8)
      g_x[i,j,k] = -(Phi[i+1,j,k] - Phi[i-1,j,k]) / (2 dx_l), same for y, z,
  where a neighbour the level itself cannot supply is taken as follows:

  * method A (Eq. A.1; L90): a neighbour outside a FINE grid (level l > 0) is the
    ghost value interpolated from the parent level with Eq. 3-6 (L64-L76): the ghost cell
    with fine index f (-1 or N along one axis) has parent p = N/4 + floor(f/2) and
    child-offset sign s = +1 (f odd) / -1 (f even) per axis, value
    3/4 Phi_c[p] + 1/4 Phi_c[p+s]   (the paper's 2-point diagonal formula, reading 6);
  * method B (Eq. A.2; L90 "the first simple method"): a neighbour of a COARSE cell
    that lies under the finer grid (inside the cavity [N/4, 3N/4)^3) is replaced by the
    arithmetic mean of the potentials of its 8 children on level l+1 (the 2-D list of four
    children at L393 is garbled; 3-D = all eight, reading A2);
  * the outer boundary of level 0 has no neighbour at all (the convolution method needs no
    boundary values, L164): second-order one-sided difference
    g_x[0] = -(-3 Phi[0] + 4 Phi[1] - Phi[2]) / (2 dx)   (paper-silent, reading A1).

Output layout: g[level, component (x, y, z), k (z), j (y), i (x)].
"""
from __future__ import annotations

import numpy as np


def child_mean(phi_fine: np.ndarray) -> np.ndarray:
    """(N/2)^3 array: arithmetic mean of the 8 children of every parent cell (Eq. A.2)."""
    N = phi_fine.shape[0]
    H = N // 2
    return phi_fine.reshape(H, 2, H, 2, H, 2).mean(axis=(1, 3, 5))


def with_children(phi_l: np.ndarray, phi_finer: np.ndarray | None) -> np.ndarray:
    """Level potential in which the cells under the finer grid carry their children's mean (method B)."""
    out = np.array(phi_l, dtype=np.float64, copy=True)
    if phi_finer is not None:
        N = out.shape[0]
        Q = N // 4
        out[Q:3 * Q, Q:3 * Q, Q:3 * Q] = child_mean(phi_finer)
    return out


def ghost_value(phi_coarse: np.ndarray, fk: int, fj: int, fi: int) -> float:
    """Eq. 3-6 value at the fine-index position (fk, fj, fi) (any of them may be -1 or N)."""
    N = phi_coarse.shape[0]
    Q = N // 4
    p = [Q + (f // 2) for f in (fk, fj, fi)]            # floor division: -1 // 2 = -1
    s = [1 if (f % 2) else -1 for f in (fk, fj, fi)]    # python: -1 % 2 = 1 (odd)
    return 0.75 * phi_coarse[p[0], p[1], p[2]] + 0.25 * phi_coarse[p[0] + s[0], p[1] + s[1], p[2] + s[2]]


def padded_level(phi: np.ndarray, l: int) -> np.ndarray:
    """(N+2)^3 array: the level's potential (method B applied) with one layer of ghosts on every
    face (method A); corners/edges of the padding are never used by the stencil and stay NaN.
    On level 0 the ghost layer is set so that the central formula equals the one-sided one:
    ghost = 3 Phi[0] - 3 Phi[1] + Phi[2]."""
    L, N = phi.shape[0], phi.shape[1]
    core = with_children(phi[l], phi[l + 1] if l + 1 < L else None)
    P = np.full((N + 2, N + 2, N + 2), np.nan)
    P[1:-1, 1:-1, 1:-1] = core
    if l == 0:
        for ax in range(3):
            c = np.moveaxis(core, ax, 0)
            lo = 3.0 * c[0] - 3.0 * c[1] + c[2]
            hi = 3.0 * c[-1] - 3.0 * c[-2] + c[-3]
            Pm = np.moveaxis(P, ax, 0)
            Pm[0, 1:-1, 1:-1] = lo
            Pm[-1, 1:-1, 1:-1] = hi
    else:
        pc = phi[l - 1]                                  # Eq. 3-6 take the parent level's potential as it is
        Q = N // 4
        t = np.arange(N)                                 # fine index along a tangential axis
        pt, st = Q + t // 2, np.where(t % 2 == 1, 1, -1)
        for ax in range(3):
            for f, slot in ((-1, 0), (N, N + 1)):
                pf, sf = Q + (f // 2), (1 if f % 2 else -1)   # python: -1 // 2 = -1, -1 % 2 = 1
                near, far = [None] * 3, [None] * 3       # index arrays of the 3/4 and the 1/4 parent
                o1, o2 = [a for a in range(3) if a != ax]
                near[ax], far[ax] = pf, pf + sf
                near[o1], far[o1] = pt[:, None], (pt + st)[:, None]
                near[o2], far[o2] = pt[None, :], (pt + st)[None, :]
                face = 0.75 * pc[near[0], near[1], near[2]] + 0.25 * pc[far[0], far[1], far[2]]
                pos = [slice(1, -1)] * 3
                pos[ax] = slot
                P[tuple(pos)] = face                     # face[u, v]: u along o1, v along o2 (o1 < o2)
    return P


def acceleration(phi: np.ndarray, dx0: float) -> np.ndarray:
    """g[l, c] for every level; phi is [L, N, N, N] (z, y, x), dx_l = dx0 / 2^l."""
    phi = np.asarray(phi, dtype=np.float64)
    L, N = phi.shape[0], phi.shape[1]
    g = np.empty((L, 3, N, N, N))
    for l in range(L):
        dx = dx0 / 2.0 ** l
        P = padded_level(phi, l)
        g[l, 0] = -(P[1:-1, 1:-1, 2:] - P[1:-1, 1:-1, :-2]) / (2.0 * dx)
        g[l, 1] = -(P[1:-1, 2:, 1:-1] - P[1:-1, :-2, 1:-1]) / (2.0 * dx)
        g[l, 2] = -(P[2:, 1:-1, 1:-1] - P[:-2, 1:-1, 1:-1]) / (2.0 * dx)
    return g
