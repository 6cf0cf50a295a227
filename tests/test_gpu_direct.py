"""Parity of cm_direct_sum (CUDA, through the C ABI) against oracle.direct_sum (Eq. B.7): bar 1e-11 max |Phi|
(same operations, different summation order over N^3 same-sign terms)."""
import numpy as np
import pytest

import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _plan(N, L, dx0, G=1.0):
    import paper_2301_06763_b200 as pkg
    pkg.build()
    return pkg, pkg.Plan(N, L, dx0, G=G)


@pytest.mark.parametrize("src,dst", [(1, 0), (2, 0), (2, 1)])
def test_whole_grid_at_N16(src, dst):
    N, L, dx0 = 16, 3, 0.11
    rng = np.random.default_rng(10 * src + dst)
    rho = rng.standard_normal((L, N, N, N))
    pkg, plan = _plan(N, L, dx0, G=1.7)
    got = plan.direct_sum(torch.from_numpy(rho).cuda(), src, dst).cpu().numpy()
    ref = oracle.direct_sum(rho[src], dx0, src, dst, G=1.7)
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()
    plan.close()


def test_sampled_targets_at_N32_the_size_the_paper_names():
    """direct summation pays off for N <= 32."""
    N, L, dx0 = 32, 3, 2.0 / 32
    rng = np.random.default_rng(32)
    rho = rng.random((L, N, N, N))
    pkg, plan = _plan(N, L, dx0)
    got = plan.direct_sum(torch.from_numpy(rho).cuda(), 2, 0).cpu().numpy()
    tg = [(0, 0, 0), (31, 31, 31), (15, 16, 16), (16, 15, 17), (3, 29, 11)]
    ref = oracle.direct_sum(rho[2], dx0, 2, 0, targets=tg)
    for t, r in zip(tg, ref):
        assert abs(got[t] - r) <= 1e-11 * np.abs(got).max()
    plan.close()


def test_point_mass_closed_form_and_error_codes():
    N, L, dx0 = 16, 3, 0.125
    rho = np.zeros((L, N, N, N))
    rho[2][3, 9, 12] = 2.5
    pkg, plan = _plan(N, L, dx0)
    d = torch.from_numpy(rho).cuda()
    got = plan.direct_sum(d, 2, 0).cpu().numpy()
    dxs = dx0 / 4
    ps = [(s + 0.5 - N / 2) * dxs for s in (3, 9, 12)]
    for t in [(0, 0, 0), (7, 8, 8), (15, 0, 15)]:
        pt = [(v + 0.5 - N / 2) * dx0 for v in t]
        r = np.sqrt(sum((a - b) ** 2 for a, b in zip(pt, ps)))
        assert abs(got[t] + 2.5 * dxs ** 3 / r) <= 1e-14 * abs(got[t])
    out = torch.empty(N, N, N, dtype=torch.float64, device="cuda")
    for bad in [(0, 0), (0, 1), (3, 0), (1, -1)]:
        with pytest.raises(pkg.CMError):
            pkg.cm_direct_sum(plan.handle, d.data_ptr(), bad[0], bad[1], out.data_ptr(), 0)
    plan.close()
