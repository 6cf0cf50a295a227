"""Pins of oracle.direct_sum (Eq. B.7)."""
import numpy as np

import oracle


def test_single_fine_cell_is_the_point_mass_potential():
    N, dx0, G = 16, 0.125, 1.3
    rho = np.zeros((N, N, N))
    src = (3, 9, 12)
    rho[src] = 2.5
    phi = oracle.direct_sum(rho, dx0, 2, 0, G=G)
    dxs = dx0 / 4
    ps = [(s + 0.5 - N / 2) * dxs for s in src]
    for t in [(0, 0, 0), (15, 15, 15), (7, 8, 8), (8, 7, 9)]:
        pt = [(v + 0.5 - N / 2) * dx0 for v in t]
        r = np.sqrt(sum((a - b) ** 2 for a, b in zip(pt, ps)))
        assert abs(phi[t] - (-G * 2.5 * dxs ** 3 / r)) <= 1e-15 * abs(phi[t])


def test_targets_match_the_full_evaluation_and_axes_are_not_transposed():
    rng = np.random.default_rng(2)
    N = 8
    rho = rng.random((N, N, N))
    full = oracle.direct_sum(rho, 0.25, 1, 0)
    tg = [(0, 1, 2), (7, 0, 3), (4, 4, 4)]
    some = oracle.direct_sum(rho, 0.25, 1, 0, targets=tg)
    assert all(abs(full[t] - v) <= 1e-15 * abs(v) for t, v in zip(tg, some))
    rho = np.zeros((N, N, N))
    rho[:, :, N - 1] = 1.0                       # mass at large +x only
    phi = oracle.direct_sum(rho, 0.25, 1, 0)
    assert abs(phi[4, 4, 7]) > abs(phi[4, 4, 0]) and abs(phi[4, 7, 4] - phi[4, 0, 4]) < 1e-12


def test_far_field_is_minus_GM_over_r_and_linear():
    rng = np.random.default_rng(3)
    N = 8
    rho = rng.random((N, N, N))
    dx0 = 1.0
    phi = oracle.direct_sum(rho, dx0, 3, 0)      # source grid is 1/8 of the coarse cell size: a point from far away
    M = rho.sum() * (dx0 / 8) ** 3
    r = np.sqrt(3) * 3.5 * dx0                   # corner cell centre
    assert abs(phi[0, 0, 0] / (-M / r) - 1) < 2e-2
    a, b = rng.random((N, N, N)), rng.random((N, N, N))
    pa, pb = oracle.direct_sum(a, dx0, 1, 0), oracle.direct_sum(b, dx0, 1, 0)
    pc = oracle.direct_sum(2 * a - 3 * b, dx0, 1, 0)
    assert np.abs(pc - (2 * pa - 3 * pb)).max() <= 1e-13 * np.abs(pc).max()


def test_consistent_with_the_doubled_grid_route_at_the_coarse_centres():
    """B.7 evaluates at the coarse cell centre, the doubled-grid route (B.1) averages the fine-resolution potential
    over the coarse cell: the two differ at second order in dx, and agree to a few per cent two cells away from
    the fine grid and better far away."""
    N, dx0 = 16, 0.125
    rng = np.random.default_rng(4)
    rho = np.zeros((2, N, N, N))
    rho[1] = rng.random((N, N, N))
    mod = oracle.solve_modified(rho, dx0)[0]     # coarse grid is empty: Phi(Omega^1) is the doubled-grid term alone
    ds = oracle.direct_sum(rho[1], dx0, 1, 0)
    far = np.ones((N, N, N), bool)
    far[2:14, 2:14, 2:14] = False
    assert np.abs(mod[far] / ds[far] - 1).max() < 5e-3
