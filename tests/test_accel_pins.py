"""Pins of the acceleration oracle (oracle/cm_accel.py) against what the paper and
the mathematics fix: Eq. 8, Eq. 3-6 (L64-L76), Eq. A.1-A.2 (L382-L393), Table 4 (L232-L238)."""
import os

import numpy as np
import pytest

import oracle
from closed_forms import ellipsoid_g, sphere_g

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _centres3(N, l, half0=1.0):
    c = -half0 / 2 ** l + (np.arange(N) + 0.5) * (2 * half0 / N / 2 ** l)
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    return X, Y, Z


def _field(N, L, f, half0=1.0):
    out = np.empty((L, N, N, N))
    for l in range(L):
        out[l] = f(*_centres3(N, l, half0))
    return out


def test_affine_potential_gives_constant_acceleration_everywhere():
    """Every ingredient (central stencil, Eq. 3-6 ghosts, child means, one-sided outer boundary) is
    exact on an affine field: g = -b on every cell of every level, interfaces included.  A wrong sign,
    a wrong parent index or a wrong dx_l fails here."""
    N, L = 16, 3
    b = np.array([0.3, -0.7, 1.1])
    phi = _field(N, L, lambda X, Y, Z: 0.5 + b[0] * X + b[1] * Y + b[2] * Z)
    g = oracle.acceleration(phi, 2.0 / N)
    for c in range(3):
        assert np.abs(g[:, c] + b[c]).max() < 1e-13


def test_components_are_not_transposed():
    N, L = 16, 2
    phi = _field(N, L, lambda X, Y, Z: 2.0 * X + 0.0 * Y + 0.0 * Z)
    g = oracle.acceleration(phi, 2.0 / N)
    assert np.abs(g[:, 0] + 2.0).max() < 1e-13 and np.abs(g[:, 1]).max() < 1e-13 and np.abs(g[:, 2]).max() < 1e-13


def test_quadratic_potential_interior_and_outer_boundary():
    """Central differences and the second-order one-sided boundary formula are exact on quadratics:
    on the finest level away from the ghosts, and on level 0 away from the cavity."""
    N, L = 16, 2
    phi = _field(N, L, lambda X, Y, Z: X * X + 2.0 * Y * Y - 0.5 * Z * Z)
    g = oracle.acceleration(phi, 2.0 / N)
    X, Y, Z = _centres3(N, 1)
    s = slice(1, N - 1)
    assert np.abs(g[1, 0][s, s, s] + 2 * X[s, s, s]).max() < 1e-12
    assert np.abs(g[1, 2][s, s, s] - Z[s, s, s]).max() < 1e-12
    X, Y, Z = _centres3(N, 0)
    far = slice(0, N // 4 - 1)          # cells whose neighbours are all uncovered, outer boundary included
    assert np.abs(g[0, 0][far, far, far] + 2 * X[far, far, far]).max() < 1e-12
    assert np.abs(g[0, 1][far, far, far] + 4 * Y[far, far, far]).max() < 1e-12


def test_ghost_value_follows_eq3_6_table():
    """tests/golden/eq3_6_interpolation.txt: on the left x interface the ghost takes
    0.75 of its parent (ib) and 0.25 of (ib+1, kb+-1, lb+-1), + for odd, - for even tangential index
    (the paper's ghost-inclusive index k = our fine index + 2, same parity)."""
    N = 16
    Q = N // 4
    rows = [l.split() for l in open(os.path.join(GOLD, "eq3_6_interpolation.txt")) if not l.startswith("#")]
    for k_odd, l_odd, wn, wf, dk, dl in rows:
        fj = 5 if int(k_odd) else 4       # y index plays the paper's k, z index its l
        fk = 7 if int(l_odd) else 6
        for probe in range(3):            # unit impulses on the two cells the formula names
            phi_c = np.zeros((N, N, N))
            near = (Q + fk // 2, Q + fj // 2, Q - 1)
            far = (near[0] + int(dl), near[1] + int(dk), near[2] + 1)
            if probe == 0:
                phi_c[near] = 1.0
                want = float(wn)
            elif probe == 1:
                phi_c[far] = 1.0
                want = float(wf)
            else:
                phi_c[:] = 1.0
                phi_c[near] = phi_c[far] = 0.0
                want = 0.0
            assert oracle.ghost_value(phi_c, fk, fj, -1) == want


def test_child_mean_is_the_arithmetic_average_of_eq_a2():
    rng = np.random.default_rng(3)
    f = rng.standard_normal((8, 8, 8))
    m = oracle.child_mean(f)
    assert m.shape == (4, 4, 4)
    assert abs(m[1, 2, 3] - f[2:4, 4:6, 6:8].sum() / 8.0) < 1e-15


def test_mirror_antisymmetry():
    rng = np.random.default_rng(4)
    phi = rng.standard_normal((3, 16, 16, 16))
    g = oracle.acceleration(phi, 0.125)
    gm = oracle.acceleration(phi[:, :, :, ::-1].copy(), 0.125)
    assert np.abs(gm[:, 0][:, :, :, ::-1] + g[:, 0]).max() < 1e-12
    assert np.abs(gm[:, 1][:, :, :, ::-1] - g[:, 1]).max() < 1e-12


def test_homogeneous_sphere_acceleration():
    """|g| = 4/3 pi G rho r inside, G M / r^2 outside (named at PAPER.md:L78), on the potential of the
    nested solve: mean error on uncovered cells below 1 % at N = 32, m = 3."""
    import workloads
    N, L = 32, 3
    rho = workloads.make_rho(1, N=N, L=L)
    phi = oracle.solve(rho, 2.0 / N, method="fft")
    g = oracle.acceleration(phi, 2.0 / N)
    Q = N // 4
    errs = []
    for l in range(L):
        X, Y, Z = _centres3(N, l)
        an = sphere_g(X, Y, Z, 0.3, 1.0)
        num = np.sqrt((g[l] ** 2).sum(axis=0))
        m = np.ones((N, N, N), bool)
        if l < L - 1:
            m[Q:3 * Q, Q:3 * Q, Q:3 * Q] = False
        errs.append((np.abs(num - an) / an)[m])
    e = np.concatenate(errs)
    assert e.mean() < 0.01


@pytest.mark.slow
def test_paper_table4_ellipsoid_soft_pin():
    """tests/golden/table4_acceleration.txt: ellipsoid 0.5:1:1, [-2.25,2.25]^3, N=128,
    m=4: max 1.74 %, mean 0.05 %, sigma 0.12 %.  Evaluated as the paper does for its error plots (L206: "the
    vertical x-z plane passing through the coordinate center"), on the cells not covered by a finer grid.
    This reading reproduces the printed maximum to three digits (1.740 %); mean and sigma are soft (x2):
    the paper does not say which cells enter them."""
    row = [l.split() for l in open(os.path.join(GOLD, "table4_acceleration.txt")) if l.startswith("ellipsoid")][0]
    gmax, gmean, gsig = (float(v) for v in row[1:])
    N, L, half0 = 128, 4, 2.25
    ax = (0.5, 1.0, 1.0)
    rho = _field(N, L, lambda X, Y, Z: ((X / ax[0]) ** 2 + (Y / ax[1]) ** 2 + (Z / ax[2]) ** 2 <= 1.0) * 1.0, half0)
    phi = oracle.solve(rho, 2 * half0 / N, method="fft")
    g = oracle.acceleration(phi, 2 * half0 / N)
    Q = N // 4
    e = []
    for l in range(L):
        X, Y, Z = _centres3(N, l, half0)
        gx, gy, gz = ellipsoid_g(X, Y, Z, ax, 1.0)
        an = np.sqrt(gx * gx + gy * gy + gz * gz)
        num = np.sqrt((g[l] ** 2).sum(axis=0))
        el = 100 * np.abs((num - an) / an)
        m = np.ones((N, N, N), bool)
        if l < L - 1:
            m[Q:3 * Q, Q:3 * Q, Q:3 * Q] = False
        e.append(el[:, N // 2, :][m[:, N // 2, :]])
    e = np.concatenate(e)
    assert abs(e.max() - gmax) < 0.02 * gmax
    assert gmean / 2 < e.mean() < gmean * 2
    assert gsig / 2 < e.std() < gsig * 2


def test_paper_table4_binary_pin():
    """tests/golden/table4_acceleration.txt, binary column (set-up L78: spheres of radius 0.2 at
    x = -0.5 / +0.5, mass ratio 2:1, [-2.25,2.25]^3, N = 128, m = 4): max 9.4 %, mean 0.38 %, sigma 0.29 %.  On the
    cells not covered by a finer grid the oracle gives max 9.402 % and mean 0.383 % over all of them, sigma 0.295 % on
    the plane through the two centres (the plane the paper plots; over all cells 0.179 %) — the printed values to
    their last digit.  The analytic field is the vector sum of the two spheres (Stone & Norman 1992, cited L78)."""
    row = [l.split() for l in open(os.path.join(GOLD, "table4_acceleration.txt")) if l.startswith("binary")][0]
    gmax, gmean, gsig = (float(v) for v in row[1:])
    N, L, half0, R = 128, 4, 2.25, 0.2
    cen = ((-0.5, 0.0, 0.0), (0.5, 0.0, 0.0))
    dens = (2.0, 1.0)
    rho = _field(N, L, lambda X, Y, Z: sum(d * ((X - c[0]) ** 2 + Y ** 2 + Z ** 2 <= R * R) for c, d in zip(cen, dens)), half0)
    phi = oracle.solve(rho, 2 * half0 / N, method="fft")
    g = oracle.acceleration(phi, 2 * half0 / N)
    Q = N // 4
    e_all, e_plane = [], []
    for l in range(L):
        X, Y, Z = _centres3(N, l, half0)
        a = np.zeros((3, N, N, N))
        for c, d in zip(cen, dens):
            dx, dy, dz = X - c[0], Y - c[1], Z - c[2]
            r = np.sqrt(dx * dx + dy * dy + dz * dz)
            mag = sphere_g(X, Y, Z, R, d, centre=c)
            a -= mag * np.stack((dx, dy, dz)) / r
        an = np.sqrt((a ** 2).sum(axis=0))
        num = np.sqrt((g[l] ** 2).sum(axis=0))
        el = 100 * np.abs((num - an) / an)
        m = np.ones((N, N, N), bool)
        if l < L - 1:
            m[Q:3 * Q, Q:3 * Q, Q:3 * Q] = False
        e_all.append(el[m])
        e_plane.append(el[:, N // 2, :][m[:, N // 2, :]])
    e_all, e_plane = np.concatenate(e_all), np.concatenate(e_plane)
    assert abs(e_all.max() - gmax) < 0.02 * gmax
    assert abs(e_all.mean() - gmean) < 0.05 * gmean
    assert abs(e_plane.std() - gsig) < 0.05 * gsig
