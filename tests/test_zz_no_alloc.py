"""cm_direct_sum_static — Eq. B.7 with its scratch in a static __device__ array, for callers that
cannot call cudaMalloc — against the existing path (cm_direct_sum, scratch in the plan's workspace), on two calls in a
row that share the array.  Collected last (test_zz_*): the suite runs with pytest -x."""
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

TOL = 1e-11   # the bar of every floating-point parity test here: relative to max |Phi|


def _existing_path(pkg, rho_levels, N, L, dx0, src, dst, G):
    plan = pkg.Plan(N, L, dx0, G=G)
    ref = plan.direct_sum(rho_levels, src, dst).clone()
    torch.cuda.synchronize()
    plan.close()
    return ref


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_the_existing_path_on_two_calls_in_a_row():
    import paper_2301_06763_b200 as pkg
    pkg.build()
    pkg.cm_direct_sum_static_setup()
    # call 1 fills all 16 x 32^3 entries of the array; call 2 (smaller grid, other levels and sign mix) runs right
    # behind it on the same stream and must not see any of them
    cases = [dict(N=32, L=3, dx0=2.0 / 32, src=2, dst=0, G=1.0, seed=1),
             dict(N=20, L=3, dx0=0.37, src=2, dst=1, G=1.7, seed=2)]
    rhos, refs, outs = [], [], []
    for c in cases:
        rng = np.random.default_rng(c["seed"])
        rho = rng.standard_normal((c["L"], c["N"], c["N"], c["N"])) + (0.5 if c["seed"] == 1 else 0.0)
        d = torch.from_numpy(rho).cuda()
        rhos.append(d)
        refs.append(_existing_path(pkg, d, c["N"], c["L"], c["dx0"], c["src"], c["dst"], c["G"]))
        outs.append(torch.full((c["N"],) * 3, float("nan"), dtype=torch.float64, device="cuda"))
    torch.cuda.synchronize()
    for rep in range(2):                      # the pair twice: the second round starts from the first round's leftovers
        for o in outs:
            o.fill_(float("nan"))
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for c, d, o in zip(cases, rhos, outs):
            dxs, dxd = c["dx0"] / 2 ** c["src"], c["dx0"] / 2 ** c["dst"]
            pkg.direct_sum_static(d[c["src"]], dxs, dxd, o, G=c["G"])
        torch.cuda.synchronize()
        free1 = torch.cuda.mem_get_info()[0]
        if rep == 1:                          # (the first launch of a kernel may load its module)
            assert free1 == free0, f"device memory in use changed by {free0 - free1} bytes across two calls"
        for c, o, ref in zip(cases, outs, refs):
            assert torch.isfinite(o).all()
            err = (o - ref).abs().max().item() / ref.abs().max().item()
            assert err <= TOL, (c, rep, err)
        assert pkg.cm_static_last_error() == ""


@pytest.mark.gpu
def test_static_scratch_entry_point_rejects_what_does_not_fit():
    import paper_2301_06763_b200 as pkg
    pkg.build()
    N = pkg.CM_STATIC_MAX_N + 4
    d = torch.zeros(N, N, N, dtype=torch.float64, device="cuda")
    o = torch.full_like(d, 7.0)
    with pytest.raises(pkg.CMError) as ei:
        pkg.direct_sum_static(d, 0.5, 1.0, o)
    assert ei.value.code == pkg.CM_EINVAL
    assert "CM_STATIC_MAX_N = 32" in str(ei.value) and "N = 36" in str(ei.value)
    torch.cuda.synchronize()
    assert (o == 7.0).all()                   # nothing ran
    ok = torch.zeros(16, 16, 16, dtype=torch.float64, device="cuda")
    for bad in [dict(dx_src=0.0, dx_dst=1.0), dict(dx_src=0.5, dx_dst=-1.0), dict(dx_src=float("nan"), dx_dst=1.0)]:
        with pytest.raises(pkg.CMError) as ei:
            pkg.direct_sum_static(ok, out=torch.empty_like(ok), **bad)
        assert ei.value.code == pkg.CM_EINVAL
    with pytest.raises(pkg.CMError):
        pkg.cm_direct_sum_static(16, 0.5, 1.0, 1.0, 0, ok.data_ptr(), 0)


def test_size_limit_is_checked_before_any_cuda_call():
    """No GPU needed: the arguments are validated first, and the error text names the limit."""
    import paper_2301_06763_b200 as pkg
    pkg.build()
    with pytest.raises(pkg.CMError) as ei:
        pkg.cm_direct_sum_static(48, 0.5, 1.0, 1.0, 256, 512, 0)     # never dereferenced
    assert ei.value.code == pkg.CM_EINVAL and "exceeds CM_STATIC_MAX_N = 32" in str(ei.value)
    assert "CM_STATIC_MAX_N = 32" in pkg.cm_static_last_error()
    hdr = open(os.path.join(os.path.dirname(pkg.__file__), "..", "include", "cm.h")).read()
    assert "#define CM_STATIC_MAX_N 32" in hdr and pkg.CM_STATIC_MAX_N == 32
