"""Closed-form potentials used to pin the oracle (test-only; G explicit).

* homogeneous sphere and homogeneous ellipsoid: the two analytic solutions the
  paper tests against (Chandrasekhar 1969 / Stone & Norman 1992);
* truncated (1+(r/a)^2)^-1 envelope and Gaussian clump: textbook spherical
  solutions for the config 3/4 shapes (SURVEY.md §8c "extra closed forms").
"""
from __future__ import annotations

import numpy as np
from scipy.special import erf


def sphere_phi(x, y, z, R, rho, centre=(0.0, 0.0, 0.0), G=1.0):
    """Phi = -2 pi G rho (R^2 - r^2/3) inside, -G M / r outside, M = 4/3 pi R^3 rho."""
    r = np.sqrt((x - centre[0]) ** 2 + (y - centre[1]) ** 2 + (z - centre[2]) ** 2)
    M = 4.0 / 3.0 * np.pi * R ** 3 * rho
    with np.errstate(divide="ignore"):
        out = np.where(r <= R, -2.0 * np.pi * G * rho * (R * R - r * r / 3.0), -G * M / r)
    return out


_GL_X, _GL_W = np.polynomial.legendre.leggauss(96)
_GL_X = 0.5 * (_GL_X + 1.0)      # nodes on (0, 1)
_GL_W = 0.5 * _GL_W


def _ellipsoid_lambda(x2, y2, z2, a2):
    """Positive root of sum x_i^2/(a_i^2 + lam) = 1 (0 for interior points)."""
    f0 = x2 / a2[0] + y2 / a2[1] + z2 / a2[2] - 1.0
    lam = np.zeros_like(f0)
    out = f0 > 0
    if not np.any(out):
        return lam
    X, Y, Z = x2[out], y2[out], z2[out]
    l = np.zeros_like(X)
    for _ in range(200):  # Newton from the left on a convex decreasing function: monotone
        d0, d1, d2 = a2[0] + l, a2[1] + l, a2[2] + l
        f = X / d0 + Y / d1 + Z / d2 - 1.0
        fp = -(X / d0 ** 2 + Y / d1 ** 2 + Z / d2 ** 2)
        step = -f / fp
        l = l + step
        if np.all(np.abs(step) <= 1e-15 * (1.0 + l)):
            break
    lam[out] = l
    return lam


def ellipsoid_phi(x, y, z, semi_axes, rho, G=1.0):
    """Chandrasekhar's homogeneous-ellipsoid potential (body frame, centred):

    Phi = -pi G rho a1 a2 a3 int_lam^inf [1 - sum x_i^2/(a_i^2+u)] du / sqrt(prod (a_i^2+u)),
    lam = 0 inside.  Quadrature: u = lam + amax^2 (w^-2 - 1), w in (0, 1].
    """
    x, y, z = np.broadcast_arrays(np.asarray(x, float), np.asarray(y, float), np.asarray(z, float))
    shape = x.shape
    x2, y2, z2 = (x.ravel() ** 2, y.ravel() ** 2, z.ravel() ** 2)
    a2 = np.asarray(semi_axes, float) ** 2
    amax2 = a2.max()
    lam = _ellipsoid_lambda(x2, y2, z2, a2)
    acc = np.zeros_like(lam)
    for w, wt in zip(_GL_X, _GL_W):
        u = lam + amax2 * (1.0 / (w * w) - 1.0)
        d0, d1, d2 = a2[0] + u, a2[1] + u, a2[2] + u
        integrand = (1.0 - x2 / d0 - y2 / d1 - z2 / d2) / np.sqrt(d0 * d1 * d2)
        acc += wt * integrand * (2.0 * amax2 / w ** 3)
    pref = -np.pi * G * rho * np.sqrt(a2.prod())
    return (pref * acc).reshape(shape)


def envelope_phi(r, rho0, a, Rt, G=1.0):
    """rho = rho0/(1+r^2/a^2) for r <= Rt, else 0.
    M(<r) = 4 pi rho0 a^2 (r - a atan(r/a));  for r <= Rt
    Phi = -G [ M(<r)/r + 2 pi rho0 a^2 ln((a^2+Rt^2)/(a^2+r^2)) ],  -G M(<Rt)/r outside."""
    r = np.asarray(r, float)
    M = lambda s: 4.0 * np.pi * rho0 * a * a * (s - a * np.arctan(s / a))
    inner = -G * (M(r) / r + 2.0 * np.pi * rho0 * a * a * np.log((a * a + Rt * Rt) / (a * a + r * r)))
    return np.where(r <= Rt, inner, -G * M(Rt) / r)


def gaussian_phi(s, A, sigma, G=1.0):
    """rho = A exp(-s^2 / 2 sigma^2): M = A (2 pi)^(3/2) sigma^3, Phi = -G M erf(s/(sqrt2 sigma))/s."""
    s = np.asarray(s, float)
    M = A * (2.0 * np.pi) ** 1.5 * sigma ** 3
    return -G * M * erf(s / (np.sqrt(2.0) * sigma)) / s


def sphere_g(x, y, z, R, rho, centre=(0.0, 0.0, 0.0), G=1.0):
    """|g| of a homogeneous sphere: 4/3 pi G rho r inside, G M / r^2 outside."""
    r = np.sqrt((x - centre[0]) ** 2 + (y - centre[1]) ** 2 + (z - centre[2]) ** 2)
    M = 4.0 / 3.0 * np.pi * R ** 3 * rho
    with np.errstate(divide="ignore"):
        return np.where(r <= R, 4.0 / 3.0 * np.pi * G * rho * r, G * M / (r * r))


def ellipsoid_g(x, y, z, semi_axes, rho, G=1.0):
    """Acceleration components of Chandrasekhar's homogeneous ellipsoid: the derivative of
    ellipsoid_phi (the lambda-dependence drops out because the integrand vanishes at u = lambda):
    g_i = -2 pi G rho a1 a2 a3 x_i int_lam^inf du / ((a_i^2+u) sqrt(prod (a_j^2+u)))."""
    x, y, z = np.broadcast_arrays(np.asarray(x, float), np.asarray(y, float), np.asarray(z, float))
    shape = x.shape
    xs = (x.ravel(), y.ravel(), z.ravel())
    a2 = np.asarray(semi_axes, float) ** 2
    amax2 = a2.max()
    lam = _ellipsoid_lambda(xs[0] ** 2, xs[1] ** 2, xs[2] ** 2, a2)
    acc = [np.zeros_like(lam) for _ in range(3)]
    for w, wt in zip(_GL_X, _GL_W):
        u = lam + amax2 * (1.0 / (w * w) - 1.0)
        d = (a2[0] + u, a2[1] + u, a2[2] + u)
        delta = np.sqrt(d[0] * d[1] * d[2])
        for i in range(3):
            acc[i] += wt * (2.0 * amax2 / w ** 3) / (d[i] * delta)
    pref = -2.0 * np.pi * G * rho * np.sqrt(a2.prod())
    return tuple((pref * xs[i] * acc[i]).reshape(shape) for i in range(3))
