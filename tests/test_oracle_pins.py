"""Pins for the oracle: everything here compares oracle/ against something that is
NOT the oracle — closed forms, library routines, brute force, values printed in the
paper — so that a dropped term, wrong sign/index or transposed operand fails a test.
CPU only (-m "not gpu")."""
import os

import numpy as np
import pytest
from scipy.signal import fftconvolve

import oracle
import workloads
from closed_forms import ellipsoid_phi, sphere_phi, envelope_phi, gaussian_phi

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


# ---------------------------------------------------------------- Eq. 13: I0
def test_I0_against_smooth_quadrature():
    """I0 = int_{[-1/2,1/2]^3} d^3u/|u|.  In spherical coordinates the radial integral
    gives R(Omega)^2/2 with R the distance to the cube surface; over the cone of one
    face, with (u,v) = (nx/nz, ny/nz), this is 3 * int_0^1 int_0^1 du dv / sqrt(1+u^2+v^2)
    — a smooth integrand, so Gauss-Legendre converges to rounding."""
    x, w = np.polynomial.legendre.leggauss(40)
    x = 0.5 * (x + 1)
    w = 0.5 * w
    U, V = np.meshgrid(x, x)
    val = 3.0 * np.sum(np.outer(w, w) / np.sqrt(1 + U * U + V * V))
    assert abs(oracle.I0() - val) < 1e-14
    assert abs(oracle.I0() - 2.3800773639795) < 1e-12  # SURVEY.md §8 quotes this value


# ---------------------------------------------------------------- the oracle's FFT
@pytest.mark.parametrize("n", [2, 8, 32, 256])
def test_fft1d_against_numpy_and_naive_dft(n):
    rng = np.random.default_rng(n)
    z = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    f = oracle.fft1d(z, -1)
    assert np.abs(f - np.fft.fft(z)).max() < 1e-12 * np.abs(f).max()
    assert np.abs(f - oracle.dft_naive(z, -1)).max() < 1e-12 * np.abs(f).max()
    b = oracle.fft1d(f, +1) / n
    assert np.abs(b - z).max() < 1e-13
    # sign convention: a pure tone exp(+2 pi i j/n) lands in bin 1 of the forward transform
    tone = np.exp(2j * np.pi * np.arange(n) / n)
    ft = oracle.fft1d(tone, -1)
    assert abs(ft[1 % n] - n) < 1e-10 and (n < 3 or abs(ft[n - 1]) < 1e-10)


# ---------------------------------------------------------------- Eq. 10: point source
@pytest.mark.parametrize("method", ["direct", "fft"])
@pytest.mark.parametrize("src", [(0, 0, 0), (7, 7, 7), (7, 0, 3), (2, 5, 7), (0, 7, 0)])
def test_single_cell_source_is_inverse_distance(method, src):
    """One non-zero cell, L=1: Phi[t] = -G rho dx^2 / |t-s| (Eq. 10) and
    Phi[s] = -G rho dx^2 I0 (Eq. 13).  Sources in the corners catch wrap-around /
    off-by-one errors of the doubled mesh (Fig. 4)."""
    N, dx, G, rho0 = 8, 0.37, 1.7, 2.5
    rho = np.zeros((1, N, N, N))
    rho[0][src] = rho0
    phi = oracle.solve(rho, dx, G=G, method=method)[0]
    k, j, i = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    d = np.sqrt((k - src[0]) ** 2.0 + (j - src[1]) ** 2.0 + (i - src[2]) ** 2.0)
    with np.errstate(divide="ignore"):
        ref = -G * rho0 * dx * dx / d
    ref[src] = -G * rho0 * dx * dx * (3 * np.log(2 + np.sqrt(3)) - np.pi / 2)
    assert _rel(phi, ref) < 1e-13


def test_axes_are_not_transposed():
    """An x-elongated source must give a potential elongated in x (i = fastest index)."""
    N = 8
    rho = np.zeros((1, N, N, N))
    rho[0, 4, 4, :] = 1.0          # a rod along x
    phi = oracle.solve(rho, 1.0, method="fft")[0]
    ref = np.zeros((N, N, N))
    I0 = oracle.I0()
    for t in np.ndindex(N, N, N):
        s = 0.0
        for i in range(N):
            d2 = (t[0] - 4) ** 2 + (t[1] - 4) ** 2 + (t[2] - i) ** 2
            s += I0 if d2 == 0 else 1.0 / np.sqrt(d2)
        ref[t] = -s
    assert _rel(phi, ref) < 1e-13
    assert abs(phi[4, 4, 0]) > abs(phi[4, 0, 4]) and abs(phi[4, 4, 0]) > abs(phi[0, 4, 4])


# ---------------------------------------------------------------- single level == textbook isolated convolution
@pytest.mark.parametrize("N", [8, 16])
def test_single_level_matches_scipy_fftconvolve_and_direct(N):
    """For L=1 the method is the Hockney-Eastwood isolated convolution of rho with
    the (2N-1)^3 kernel 1/|o| (I0 at o=0): scipy's fftconvolve is a library check."""
    rng = np.random.default_rng(5)
    rho = rng.random((1, N, N, N))
    dx, G = 0.25, 1.0
    o = np.arange(-(N - 1), N)
    K, J, I = np.meshgrid(o, o, o, indexing="ij")
    with np.errstate(divide="ignore"):
        ker = 1.0 / np.sqrt(K * K + J * J + I * I + 0.0)
    ker[N - 1, N - 1, N - 1] = 3 * np.log(2 + np.sqrt(3)) - np.pi / 2
    ref = -G * dx * dx * fftconvolve(rho[0], ker, mode="full")[N - 1:2 * N - 1, N - 1:2 * N - 1, N - 1:2 * N - 1]
    pd = oracle.solve(rho, dx, method="direct")[0]
    pf = oracle.solve(rho, dx, method="fft")[0]
    assert _rel(pd, ref) < 1e-13
    assert _rel(pf, ref) < 1e-13
    assert _rel(pf, pd) < 1e-13


def test_green_hat_is_real_and_even():
    """g is even in every axis on the rearranged doubled mesh (Fig. 4), so its
    transform is real and even — the property the CUDA path's real K-hat relies on."""
    N = 8
    gh = oracle.green_hat(N)
    assert np.abs(gh.imag).max() < 1e-12 * np.abs(gh.real).max()
    n = 2 * N
    idx = (-np.arange(n)) % n
    assert np.abs(gh - gh[idx][:, idx][:, :, idx]).max() < 1e-11 * np.abs(gh).max()
    assert np.abs(gh - gh[idx]).max() < 1e-11 * np.abs(gh).max()


# ---------------------------------------------------------------- restriction (a1)
def test_restriction_conserves_mass_and_keeps_uncovered_cells():
    N, L = 8, 3
    rng = np.random.default_rng(1)
    rho = rng.random((L, N, N, N))
    rb = oracle.restrict(rho)
    lo, hi = N // 4, 3 * N // 4
    assert np.array_equal(rb[L - 1], rho[L - 1])
    for l in range(L - 1):
        mask = np.zeros((N, N, N), bool)
        mask[lo:hi, lo:hi, lo:hi] = True
        assert np.array_equal(rb[l][~mask], rho[l][~mask])                # outside the cavity: untouched
        dxc, dxf = 1.0 / (1 << l), 1.0 / (1 << (l + 1))
        m_c = rb[l][mask].sum() * dxc ** 3
        m_f = rb[l + 1].sum() * dxf ** 3
        assert abs(m_c - m_f) < 1e-13 * m_f                               # mass conservation
    # hand-computed cell: parent (lo,lo,lo) of level L-2 = mean of fine block [0:2]^3
    assert abs(rb[L - 2][lo, lo, lo] - rho[L - 1][0:2, 0:2, 0:2].mean()) < 1e-15
    # asymmetric index check: parent (lo, lo+1, lo+2) <- fine block k 0:2, j 2:4, i 4:6
    assert abs(rb[L - 2][lo, lo + 1, lo + 2] - rho[L - 1][0:2, 2:4, 4:6].mean()) < 1e-15
    # the cascade: level 0's cavity sees level 2 through level 1
    blk = rb[1][0:2, 0:2, 0:2].mean()
    assert abs(rb[0][lo, lo, lo] - blk) < 1e-15
    const = np.full((L, N, N, N), 3.25)
    assert np.array_equal(oracle.restrict(const), const)


# ---------------------------------------------------------------- prolongation (tilde of Eq. 14)
def test_prolongation_exact_on_affine_fields():
    """Eq. 3-6 is a 2-point interpolation along the cell diagonal: exact for any
    affine field evaluated at the fine cell centres."""
    N = 8
    xc = workloads.cell_centres(N, 0)
    xf = workloads.cell_centres(N, 1)
    a, b = 0.3, np.array([1.1, -0.7, 0.45])      # (z, y, x) slopes
    Kc, Jc, Ic = np.meshgrid(xc, xc, xc, indexing="ij")
    Kf, Jf, If = np.meshgrid(xf, xf, xf, indexing="ij")
    coarse = a + b[0] * Kc + b[1] * Jc + b[2] * Ic
    fine = oracle.prolong(coarse)
    assert np.abs(fine - (a + b[0] * Kf + b[1] * Jf + b[2] * If)).max() < 1e-14


def test_prolongation_matches_paper_eq3_6_parity_table():
    """Golden fixture tests/golden/eq3_6_interpolation.txt.  The
    paper's k,l run 1..N+2 with index 1 the ghost layer, so its odd k is our odd
    0-based fine index; kb = N/4 + k/2 + 1 is our parent N/4 + f/2."""
    N = 8
    rng = np.random.default_rng(3)
    coarse = rng.random((N, N, N))
    fine = oracle.prolong(coarse)
    rows = [l.split() for l in open(os.path.join(GOLD, "eq3_6_interpolation.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 4
    for kodd, lodd, wn, wf, dk, dl in rows:
        kodd, lodd, wn, wf, dk, dl = int(kodd), int(lodd), float(wn), float(wf), int(dk), int(dl)
        for k1 in range(2, N + 2):             # paper's 1-based ghost-inclusive indices of real cells
            for l1 in range(2, N + 2):
                if (k1 % 2 != 0) != bool(kodd) or (l1 % 2 != 0) != bool(lodd):
                    continue
                fy, fz = k1 - 2, l1 - 2          # paper's k is y, l is z (i, k, l <-> x, y, z)
                kb, lb = N // 4 + k1 // 2 + 1 - 2, N // 4 + l1 // 2 + 1 - 2
                for fx in (0, 1, 4, 7):
                    i1 = fx + 2
                    ib = N // 4 + i1 // 2 + 1 - 2
                    di = +1 if i1 % 2 != 0 else -1
                    ref = wn * coarse[lb, kb, ib] + wf * coarse[lb + dl, kb + dk, ib + di]
                    assert abs(fine[fz, fy, fx] - ref) < 1e-15


# ---------------------------------------------------------------- hole / full split
def test_full_equals_hole_plus_cavity_only():
    N = 8
    rng = np.random.default_rng(7)
    rho = rng.random((N, N, N))
    cav = np.zeros_like(rho)
    lo, hi = N // 4, 3 * N // 4
    cav[lo:hi, lo:hi, lo:hi] = rho[lo:hi, lo:hi, lo:hi]
    for f in (oracle.field_direct, lambda *a: oracle.field_fft(*a)):
        full = f(rho, False, 1.0, 0.5)
        hole = f(rho, True, 1.0, 0.5)
        only = f(cav, False, 1.0, 0.5)
        assert _rel(hole + only, full) < 1e-13
        assert np.abs(f(cav, True, 1.0, 0.5)).max() == 0.0


# ---------------------------------------------------------------- whole method: invariants
def _random_nested(N, L, seed):
    rng = np.random.default_rng(seed)
    return rng.random((L, N, N, N)) * (8.0 ** np.arange(L))[:, None, None, None]


def test_direct_and_fft_paths_agree_on_nested_grid():
    rho = _random_nested(8, 3, 11)
    pd = oracle.solve(rho, 0.25, method="direct")
    pf = oracle.solve(rho, 0.25, method="fft")
    for l in range(3):
        assert _rel(pf[l], pd[l]) < 1e-13


def test_linearity_and_mirror_symmetry_and_sign():
    N, L = 8, 3
    r1, r2 = _random_nested(N, L, 1), _random_nested(N, L, 2)
    a, b = 0.7, -1.3
    p1 = oracle.solve(r1, 0.25)
    p2 = oracle.solve(r2, 0.25)
    p12 = oracle.solve(a * r1 + b * r2, 0.25)
    assert _rel(p12, a * p1 + b * p2) < 1e-13
    assert p1.max() < 0                                       # Phi <= 0 for rho >= 0
    for ax in (1, 2, 3):
        pm = oracle.solve(np.flip(r1, axis=ax), 0.25)
        assert _rel(np.flip(pm, axis=ax), p1) < 1e-13


def test_two_level_assembly_by_hand():
    """Eq. 14 for two grids: Phi(O1) = Phi^1, Phi(O2) = Phi^2 + tilde Phi^1_hole, put together
    here from the primitives with numpy indexing instead of the oracle's own loop."""
    N = 8
    rho = _random_nested(N, 2, 21)
    dx0 = 0.25
    phi = oracle.solve(rho, dx0, method="direct")
    lo, hi = N // 4, 3 * N // 4
    rb0 = rho[0].copy()
    rb0[lo:hi, lo:hi, lo:hi] = rho[1].reshape(N // 2, 2, N // 2, 2, N // 2, 2).mean(axis=(1, 3, 5))
    full0 = oracle.field_direct(rb0, False, 1.0, dx0)
    rh = rb0.copy()
    rh[lo:hi, lo:hi, lo:hi] = 0
    hole0 = oracle.field_direct(rh, False, 1.0, dx0)
    full1 = oracle.field_direct(rho[1], False, 1.0, dx0 / 2)
    assert _rel(phi[0], full0) < 1e-14
    f = np.arange(N)
    p = N // 4 + f // 2
    s = np.where(f % 2 == 1, 1, -1)
    near = hole0[np.ix_(p, p, p)]
    far = hole0[np.ix_(p + s, p + s, p + s)]
    assert _rel(phi[1], full1 + 0.75 * near + 0.25 * far) < 1e-14


def test_solve_points_equals_full_solve():
    rho = _random_nested(8, 4, 5)
    phi = oracle.solve(rho, 0.25, method="direct")
    tg = [(0, 0, 0, 0), (1, 7, 0, 3), (2, 4, 4, 4), (3, 0, 7, 1), (3, 7, 7, 7), (3, 2, 5, 0)]
    ps = oracle.solve_points(rho, 0.25, tg)
    for v, t in zip(ps, tg):
        assert abs(v - phi[t]) < 1e-13 * np.abs(phi[t[0]]).max()


# ---------------------------------------------------------------- whole method: closed forms
def _centres3(N, l, half0=1.0):
    c = workloads.cell_centres(N, l, half0)
    return c[None, None, :], c[None, :, None], c[:, None, None]


def test_config1_homogeneous_sphere_closed_form_and_far_field():
    """Config 1 (2 x 16^3, sphere R=0.3, volume-fraction sampled).  Method error vs the
    analytic sphere: SURVEY probe mean 0.16 %, max 3.0 %."""
    rho = workloads.make_rho(1)
    N, L = 16, 2
    phi = oracle.solve(rho, 2.0 / N, method="direct")
    errs = []
    for l in range(L):
        X, Y, Z = _centres3(N, l)
        an = sphere_phi(X, Y, Z, 0.3, 1.0)
        errs.append(np.abs((phi[l] - an) / an))
    e = np.concatenate([x.ravel() for x in errs])
    assert e.mean() < 3e-3 and e.max() < 4e-2
    # far field at the corner cell of level 0: Phi -> -G M / r with M the mass on the grid
    rb = oracle.restrict(rho)
    M = rb[0].sum() * (2.0 / N) ** 3
    c = workloads.cell_centres(N, 0)
    r = np.sqrt(3 * c[0] ** 2)
    assert abs(phi[0][0, 0, 0] / (-M / r) - 1) < 1e-4


def test_oracleB_leaf_direct_sum_bounds_method_error_config1():
    """north_star's "direct triple sum over all cells of all levels".  On the finest level
    of config 1 the hole field carries no mass (sphere inside the fine grid), so the
    method and the physical leaf sum coincide; on the coarse level they differ by the
    method's own approximation (restricted monopoles), SURVEY probe: max 1.7 %."""
    rho = workloads.make_rho(1)
    phi = oracle.solve(rho, 2.0 / 16, method="direct")
    b1 = oracle.leaf_direct(rho, 1)
    b0 = oracle.leaf_direct(rho, 0)
    assert _rel(phi[1], b1) < 1e-13
    assert 1e-4 < _rel(phi[0], b0) < 3e-2


def test_config2_ellipsoid_closed_form():
    """Config 2 (4 x 32^3 oblate ellipsoid, S=4).  SURVEY probe: mean 0.08 %, max 0.85 %."""
    rho = workloads.make_rho(2)
    N, L = 32, 4
    phi = oracle.solve(rho, 2.0 / N, method="fft")
    e = []
    for l in range(L):
        X, Y, Z = _centres3(N, l)
        an = ellipsoid_phi(X, Y, Z, (0.4, 0.4, 0.2), 1.0)
        e.append(np.abs((phi[l] - an) / an).ravel())
    e = np.concatenate(e)
    assert e.mean() < 2e-3 and e.max() < 1.5e-2


def test_closed_forms_are_self_consistent():
    """The ellipsoid quadrature reduces to the sphere formula for equal axes, and the
    envelope formula solves its own Poisson problem (checked by radial quadrature)."""
    x = np.linspace(-1.5, 1.5, 13)
    X, Y, Z = np.meshgrid(x, x + 0.01, x - 0.02, indexing="ij")
    assert np.abs(ellipsoid_phi(X, Y, Z, (0.6, 0.6, 0.6), 2.0) / sphere_phi(X, Y, Z, 0.6, 2.0) - 1).max() < 1e-10
    from scipy.integrate import quad
    rho0, a, Rt = 1.3, 0.05, 1.0
    for r in (0.02, 0.3, 0.9, 1.4):
        dens = lambda s: rho0 / (1 + s * s / (a * a)) if s <= Rt else 0.0
        Min = quad(lambda s: 4 * np.pi * s * s * dens(s), 0, min(r, Rt), epsabs=1e-14, epsrel=1e-13)[0]
        outer = quad(lambda s: 4 * np.pi * s * dens(s), r, Rt, epsabs=1e-14, epsrel=1e-13)[0] if r < Rt else 0.0
        assert abs(envelope_phi(r, rho0, a, Rt) / (-(Min / r + outer)) - 1) < 1e-9
    A, sig = 3.0, 0.1
    for r in (0.05, 0.5):
        dens = lambda s: A * np.exp(-s * s / (2 * sig * sig))
        Min = quad(lambda s: 4 * np.pi * s * s * dens(s), 0, r, epsabs=1e-15, epsrel=1e-13)[0]
        outer = quad(lambda s: 4 * np.pi * s * dens(s), r, 20 * sig, epsabs=1e-15, epsrel=1e-13)[0]
        assert abs(gaussian_phi(r, A, sig) / (-(Min / r + outer)) - 1) < 1e-9


def test_error_falls_with_number_of_levels():
    """PAPER.md:L206 (Fig. 10): the convolution method's Phi error declines with m."""
    N = 16
    means = []
    for L in (1, 2, 3):
        rho = workloads.make_rho(1, N=N, L=L)
        phi = oracle.solve(rho, 2.0 / N)
        X, Y, Z = _centres3(N, L - 1)
        an = sphere_phi(X, Y, Z, 0.3, 1.0)
        inner = slice(N // 4, 3 * N // 4) if L < 3 else slice(0, N)
        # compare on the innermost region [-0.25,0.25]^3 covered by level 2
        if L == 1:
            sl = slice(6, 10)
        elif L == 2:
            sl = slice(4, 12)
        else:
            sl = slice(0, 16)
        means.append(np.abs((phi[L - 1][sl, sl, sl] - an[sl, sl, sl]) / an[sl, sl, sl]).mean())
    assert means[2] < means[1] < means[0]


@pytest.mark.slow
def test_paper_table3_ellipsoid_soft_pin():
    """Golden fixture tests/golden/table3_convolution.txt: oblate
    ellipsoid 0.5:1:1 in [-2.25,2.25]^3, N=128, m=4 -> max 0.045 %, mean 0.004 %,
    sigma 0.004 %.  The paper does not say how cells were sampled, so this is a soft
    pin: within x1.6 (cell-centre sampling; SURVEY probe 0.058 / 0.0036 / 0.0034)."""
    row = [l.split() for l in open(os.path.join(GOLD, "table3_convolution.txt")) if l.startswith("ellipsoid")][0]
    gmax, gmean, gsig = (float(v) for v in row[1:])
    N, L, half0 = 128, 4, 2.25
    ax = (0.5, 1.0, 1.0)
    rho = np.empty((L, N, N, N))
    for l in range(L):
        X, Y, Z = _centres3(N, l, half0)
        rho[l] = ((X / ax[0]) ** 2 + (Y / ax[1]) ** 2 + (Z / ax[2]) ** 2 <= 1.0) * 1.0
    phi = oracle.solve(rho, 2 * half0 / N, method="fft")
    e = []
    for l in range(L):
        X, Y, Z = _centres3(N, l, half0)
        an = ellipsoid_phi(X, Y, Z, ax, 1.0)
        e.append(100 * np.abs((phi[l] - an) / an).ravel())
    e = np.concatenate(e)
    assert gmax / 1.6 < e.max() < gmax * 1.6
    assert gmean / 1.6 < e.mean() < gmean * 1.6
    assert gsig / 1.6 < e.std() < gsig * 1.6


@pytest.mark.slow
def test_paper_table3_binary_soft_pin():
    """Golden fixture tests/golden/table3_convolution.txt, binary column (set-up L78: two
    homogeneous spheres of radius 0.2 centred at x = -0.5 and +0.5, mass ratio 2:1, domain [-2.25,2.25]^3; N = 128,
    m = 4, L200-L202): max 0.85 %, mean 0.43 %, sigma 0.078 %.  A non-axisymmetric field whose sources straddle the
    interface of grids 2 and 3.  With cell-centre sampling the oracle gives 0.839 / 0.400 / 0.049 (0.068 on the plane
    through the centres, the one the paper plots) — soft pin: max and mean within 10 %, sigma within x1.7."""
    row = [l.split() for l in open(os.path.join(GOLD, "table3_convolution.txt")) if l.startswith("binary")][0]
    gmax, gmean, gsig = (float(v) for v in row[1:])
    N, L, half0, R = 128, 4, 2.25, 0.2
    rho = np.empty((L, N, N, N))
    for l in range(L):
        X, Y, Z = _centres3(N, l, half0)
        rho[l] = 2.0 * ((X + 0.5) ** 2 + Y ** 2 + Z ** 2 <= R * R) + 1.0 * ((X - 0.5) ** 2 + Y ** 2 + Z ** 2 <= R * R)
    phi = oracle.solve(rho, 2 * half0 / N, method="fft")
    e = []
    for l in range(L):
        X, Y, Z = _centres3(N, l, half0)
        an = sphere_phi(X, Y, Z, R, 2.0, centre=(-0.5, 0.0, 0.0)) + sphere_phi(X, Y, Z, R, 1.0, centre=(0.5, 0.0, 0.0))
        e.append(100 * np.abs((phi[l] - an) / an).ravel())
    e = np.concatenate(e)
    assert abs(e.max() - gmax) < 0.10 * gmax
    assert abs(e.mean() - gmean) < 0.10 * gmean
    assert gsig / 1.7 < e.std() < gsig * 1.7
