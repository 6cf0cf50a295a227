"""The five BASELINE.json configs as seeded, synthetic density fields.

Geometry (Fig. 1): `levels` concentric N^3
Cartesian grids, level 0 = coarsest = the paper's m=1 covering [-1,1]^3; level
l has half-width 2^-l and cell size dx_l = dx0 / 2^l, dx0 = 2/N; cell centres
x_i = -2^-l + (i + 1/2) dx_l.  Array layout: rho[l, k, j, i] with i (x) fastest.

Shapes follow the paper's tests (homogeneous ellipsoid / spheres)
and BASELINE.json's config strings.  The paper measures on analytic shapes, not
on a dataset, so nothing stands in for anything else here.
"""
from __future__ import annotations

import numpy as np

SEED0 = 230106763  # SeedSequence([SEED0, config_id, level]) — SURVEY.md §8(d)

CONFIGS = {
    1: dict(N=16, L=2, name="2x16^3 homogeneous sphere R=0.3"),
    2: dict(N=32, L=4, name="4x32^3 oblate ellipsoid (0.4,0.4,0.2)"),
    3: dict(N=64, L=6, name="6x64^3 two spheres in a (1+(r/0.01)^2)^-1 envelope"),
    4: dict(N=128, L=8, name="8x128^3 rotated triaxial ellipsoid + Gaussian clump"),
    5: dict(N=256, L=10, name="10x256^3 log-normal k^-3 field x r^-2 envelope"),
}


def dx_level(N: int, level: int, half_width0: float = 1.0) -> float:
    """Cell size of level `level` (dx_m = (wR-wL)/(2^(m-1) N))."""
    return 2.0 * half_width0 / N / (1 << level)


def cell_centres(N: int, level: int, half_width0: float = 1.0) -> np.ndarray:
    """1-D array of the N cell-centre coordinates of a level (same in x, y, z)."""
    dx = dx_level(N, level, half_width0)
    return -half_width0 / (1 << level) + (np.arange(N) + 0.5) * dx


def level_rng(config_id: int, level: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([SEED0, config_id, level])))


def volume_fraction(inside, N: int, level: int, S: int, half_width0: float = 1.0) -> np.ndarray:
    """Fraction of each cell's S^3 sub-cell centres for which inside(x,y,z) holds.

    SURVEY.md §8(c) row 14: cell-centre sampling mis-states the mass by a few per
    cent at N<=32, so closed-form comparisons use supersampled volume fractions.
    """
    dx = dx_level(N, level, half_width0)
    lo = -half_width0 / (1 << level)
    f = lo + (np.arange(N * S) + 0.5) * (dx / S)
    out = np.zeros((N, N, N))
    # one z-slab of S fine planes at a time keeps memory small
    X = f[None, None, :]
    Y = f[None, :, None]
    for k in range(N):
        Z = f[k * S:(k + 1) * S][:, None, None]
        m = inside(X, Y, Z).astype(np.float64)          # (S, NS, NS)
        m = m.sum(axis=0)                               # (NS, NS)
        out[k] = m.reshape(N, S, N, S).sum(axis=(1, 3)) / float(S ** 3)
    return out


def _grid(N, level, half_width0=1.0):
    c = cell_centres(N, level, half_width0)
    return c[None, None, :], c[None, :, None], c[:, None, None]  # X, Y, Z broadcastable to [k,j,i]


def _cfg1(N, L):
    R = 0.3
    S = 8 if N <= 16 else (4 if N <= 32 else 1)
    ins = lambda x, y, z: x * x + y * y + z * z <= R * R
    return np.stack([volume_fraction(ins, N, l, S) for l in range(L)])


def _cfg2(N, L):
    a = (0.4, 0.4, 0.2)
    S = 8 if N <= 16 else (4 if N <= 32 else 1)
    ins = lambda x, y, z: (x / a[0]) ** 2 + (y / a[1]) ** 2 + (z / a[2]) ** 2 <= 1.0
    return np.stack([volume_fraction(ins, N, l, S) for l in range(L)])


def _cfg3(N, L):
    rho0, a, Rt = 1.0, 0.01, 1.0
    Rs, cx, dens = 0.05, 0.08, 1.0e3
    out = np.empty((L, N, N, N))
    for l in range(L):
        X, Y, Z = _grid(N, l)
        r2 = X * X + Y * Y + Z * Z
        rho = np.where(r2 <= Rt * Rt, rho0 / (1.0 + r2 / (a * a)), 0.0)
        for sgn in (+1.0, -1.0):
            rho = rho + dens * (((X - sgn * cx) ** 2 + Y * Y + Z * Z) <= Rs * Rs)
        out[l] = rho
    return out


def _cfg4(N, L):
    ax = (0.5, 0.3, 0.2)
    th = np.deg2rad(30.0)
    c, s = np.cos(th), np.sin(th)
    sig, peak, c0 = 0.002, 1.0e6, (0.003, 0.001, 0.0)
    out = np.empty((L, N, N, N))
    for l in range(L):
        X, Y, Z = _grid(N, l)
        # body-frame coordinates of a shape rotated by +30 deg about z
        xb = c * X + s * Y
        yb = -s * X + c * Y
        rho = 1.0 * ((xb / ax[0]) ** 2 + (yb / ax[1]) ** 2 + (Z / ax[2]) ** 2 <= 1.0)
        d2 = (X - c0[0]) ** 2 + (Y - c0[1]) ** 2 + (Z - c0[2]) ** 2
        out[l] = rho + peak * np.exp(-d2 / (2.0 * sig * sig))
    return out


def _cfg5(N, L):
    out = np.empty((L, N, N, N))
    kf = np.fft.fftfreq(N) * N
    kr = np.fft.rfftfreq(N) * N
    k2 = kf[:, None, None] ** 2 + kf[None, :, None] ** 2 + kr[None, None, :] ** 2
    with np.errstate(divide="ignore"):
        amp = np.where(k2 > 0, k2 ** (-0.75), 0.0)          # |k|^-3/2  => P(k) ~ k^-3
    for l in range(L):
        w = level_rng(5, l).standard_normal((N, N, N))
        d = np.fft.irfftn(np.fft.rfftn(w) * amp, s=(N, N, N), axes=(0, 1, 2))
        d = (d - d.mean()) / d.std()
        X, Y, Z = _grid(N, l)
        out[l] = np.exp(1.5 * d) / (X * X + Y * Y + Z * Z)
    return out


_MAKERS = {1: _cfg1, 2: _cfg2, 3: _cfg3, 4: _cfg4, 5: _cfg5}


def make_rho(config_id: int, N: int | None = None, L: int | None = None) -> np.ndarray:
    """Density on every level, float64 [L, N, N, N].  N/L override the config's size
    (same shape recipe, smaller grid) for tests that need a cheaper instance."""
    cfg = CONFIGS[config_id]
    N = cfg["N"] if N is None else N
    L = cfg["L"] if L is None else L
    return np.ascontiguousarray(_MAKERS[config_id](N, L), dtype=np.float64)
