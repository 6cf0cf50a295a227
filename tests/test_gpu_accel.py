"""Parity of cm_acceleration (CUDA, through the C ABI) against oracle.acceleration, element by element.

Both sides get the SAME potentials (the oracle's, or seeded random fields), so the comparison isolates the
stencil / ghost / child-mean arithmetic: only the summation order differs.  Bar: max |g_gpu - g_oracle| <=
1e-12 * max |g| per level and component set (the differences of potentials cancel to ~N eps)."""
import numpy as np
import pytest

import oracle
import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-12


def _gpu_accel(phi, dx0):
    import paper_2301_06763_b200 as pkg
    pkg.build()
    L, N = phi.shape[0], phi.shape[1]
    plan = pkg.Plan(N, L, dx0)
    d = torch.from_numpy(np.ascontiguousarray(phi)).cuda()
    keep = d.clone()
    g = plan.acceleration(d)
    torch.cuda.synchronize()
    assert torch.equal(d, keep), "phi_levels must not be written"
    out = g.cpu().numpy()
    plan.close()
    return out


def _assert_parity(got, ref):
    for l in range(ref.shape[0]):
        scale = np.abs(ref[l]).max()
        e = np.abs(got[l] - ref[l]).max()
        assert e <= TOL * scale, f"level {l}: {e:.3e} > {TOL} * {scale:.3e}"


@pytest.mark.parametrize("N,L", [(16, 1), (16, 2), (32, 3), (64, 4), (20, 3), (48, 2), (96, 2), (168, 2)])
def test_random_potentials(N, L):
    rng = np.random.default_rng(100 + N + L)
    phi = rng.standard_normal((L, N, N, N))
    dx0 = 0.37 / N                      # not a power of two: the division by 2 dx_l is exercised
    _assert_parity(_gpu_accel(phi, dx0), oracle.acceleration(phi, dx0))


def test_affine_potential_is_exact_on_the_gpu():
    N, L = 32, 3
    b = np.array([0.3, -0.7, 1.1])
    phi = np.empty((L, N, N, N))
    for l in range(L):
        c = -2.0 ** -l + (np.arange(N) + 0.5) * (2.0 / N / 2 ** l)
        Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
        phi[l] = 0.5 + b[0] * X + b[1] * Y + b[2] * Z
    g = _gpu_accel(phi, 2.0 / N)
    for c in range(3):
        assert np.abs(g[:, c] + b[c]).max() < 1e-12


def test_config3_potential_then_acceleration_end_to_end():
    """cm_potential -> cm_acceleration on the GPU against oracle.solve -> oracle.acceleration (config 3,
    6 x 64^3).  Here the potentials differ by rounding (~1e-15 of max |Phi|) before the differencing, so the
    bar is that of the potential (1e-11) times the amplification max|Phi| / (2 dx_l max|g_l|)."""
    import paper_2301_06763_b200 as pkg
    rho = workloads.make_rho(3)
    L, N = rho.shape[0], rho.shape[1]
    dx0 = 2.0 / N
    plan = pkg.Plan(N, L, dx0)
    phi = plan.potential(torch.from_numpy(rho).cuda())
    g = plan.acceleration(phi).cpu().numpy()
    phi_ref = oracle.solve(rho, dx0, method="fft")
    ref = oracle.acceleration(phi_ref, dx0)
    for l in range(L):
        amp = np.abs(phi_ref[l]).max() / (2 * dx0 / 2 ** l * np.abs(ref[l]).max())
        assert np.abs(g[l] - ref[l]).max() <= 1e-11 * amp * np.abs(ref[l]).max()
    plan.close()


def test_config5_full_size_sampled_and_invariants():
    """10 x 256^3 (the size bench.py times): sampled cells against the oracle's scalar formulas, face cells
    included; mirror antisymmetry in x on every cell."""
    N, L = 256, 10
    rng = np.random.default_rng(7)
    phi = rng.standard_normal((L, N, N, N))
    dx0 = 2.0 / N
    g = _gpu_accel(phi, dx0)
    Q = N // 4
    cells = [(0, 0, 0, 0), (0, N - 1, 5, 0), (0, Q - 1, Q, Q), (0, Q, Q, Q), (3, 0, 17, N - 1), (3, N - 1, N - 1, N - 1),
             (9, 0, 0, 0), (9, 100, N - 1, 3), (4, 3 * Q, 3 * Q - 1, Q), (L - 1, 128, 128, 128)]
    cells += [(int(rng.integers(0, L)), *(int(v) for v in rng.integers(0, N, 3))) for _ in range(20)]

    def val(l, k, j, i):               # the oracle's definitions, one cell at a time
        inside = all(0 <= v < N for v in (k, j, i))
        if inside:
            if l < L - 1 and all(Q <= v < 3 * Q for v in (k, j, i)):
                c = phi[l + 1][2 * (k - Q):2 * (k - Q) + 2, 2 * (j - Q):2 * (j - Q) + 2, 2 * (i - Q):2 * (i - Q) + 2]
                return float(oracle.child_mean(c)[0, 0, 0])
            return phi[l][k, j, i]
        if l > 0:
            return oracle.ghost_value(phi[l - 1], k, j, i)
        ax = [a for a, v in enumerate((k, j, i)) if not 0 <= v < N][0]
        p = [k, j, i]
        d = 1 if p[ax] < 0 else -1
        q0, q1, q2 = list(p), list(p), list(p)
        q0[ax] += d
        q1[ax] += 2 * d
        q2[ax] += 3 * d
        return 3.0 * val(l, *q0) - 3.0 * val(l, *q1) + val(l, *q2)

    for (l, k, j, i) in cells:
        dx = dx0 / 2 ** l
        ref = [-(val(l, k, j, i + 1) - val(l, k, j, i - 1)) / (2 * dx),
               -(val(l, k, j + 1, i) - val(l, k, j - 1, i)) / (2 * dx),
               -(val(l, k + 1, j, i) - val(l, k - 1, j, i)) / (2 * dx)]
        scale = np.abs(g[l]).max()
        for c in range(3):
            assert abs(g[l, c, k, j, i] - ref[c]) <= TOL * scale, (l, k, j, i, c)
    gm = _gpu_accel(np.ascontiguousarray(phi[:, :, :, ::-1]), dx0)
    for l in range(L):
        s = np.abs(g[l]).max()
        assert np.abs(gm[l, 0][:, :, ::-1] + g[l, 0]).max() <= TOL * s
        assert np.abs(gm[l, 1][:, :, ::-1] - g[l, 1]).max() <= TOL * s


def test_config5_size_every_cell_against_the_oracle():
    """10 x 256^3, every cell of every level and component (ZCH/TX/TY of k_accel differ from the N <= 64 cases):
    the numpy oracle is cheap enough for the whole grid."""
    N, L = 256, 10
    rng = np.random.default_rng(256)
    phi = rng.standard_normal((L, N, N, N))
    dx0 = 0.37 / N
    g = _gpu_accel(phi, dx0)
    ref = oracle.acceleration(phi, dx0)
    _assert_parity(g, ref)
    errs = [float(np.abs(g[l] - ref[l]).max() / np.abs(ref[l]).max()) for l in range(L)]
    print("PARITY cm_acceleration 10 x 256^3, whole grid: " + " ".join(f"{e:.2e}" for e in errs))


def test_error_codes():
    import paper_2301_06763_b200 as pkg
    plan = pkg.Plan(16, 2, 0.125)
    phi = torch.zeros(2, 16, 16, 16, dtype=torch.float64, device="cuda")
    with pytest.raises(pkg.CMError):
        pkg.cm_acceleration(plan.handle, phi.data_ptr(), phi.data_ptr(), 0)      # aliasing
    with pytest.raises(pkg.CMError):
        pkg.cm_acceleration(plan.handle, 0, phi.data_ptr(), 0)                   # null
    g = plan.acceleration(phi)
    assert float(g.abs().max()) == 0.0
    plan.close()
