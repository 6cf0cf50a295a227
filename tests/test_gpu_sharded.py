"""The level-sharded solve (cm_shard_restrict / cm_shard_forward / cm_shard_finish) on ONE GPU: every
emulated rank has its own plan, its own exchange buffers and only its own levels of rho; ranks are host threads whose
blocking mailbox stands in for NCCL send/recv, and all of them enqueue on the same CUDA stream, so no kernel ever
waits for another rank's kernel.  Same kernels, same arithmetic: the potentials must be BIT-identical to cm_potential's
(which the other parity tests hold against the oracle at 1e-11)."""
import queue
import threading

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _sharded(pkg, rho, N, L, dx0, G, world):
    from paper_2301_06763_b200.sharded import LevelShard, LibcmEngine, partition_levels
    parts = partition_levels(L, world)
    box = {(a, b): queue.Queue() for a in range(world) for b in range(world)}
    out, errs = [None] * world, []

    def rank_main(r):
        try:
            lo, hi = parts[r]
            eng = LibcmEngine(N, L, dx0, lo, hi, G=G) if hi > lo else None

            def send(t, peer):
                box[(r, peer)].put(t.clone())             # stream-ordered copy on the one stream every rank uses

            def recv(t, peer):
                t.copy_(box[(peer, r)].get(timeout=120))

            shard = LevelShard(L, r, world, eng, send, recv)
            rho_own = rho[lo:hi].clone()                  # the rank never sees the other levels
            phi_own = torch.full_like(rho_own, float("nan"))
            for _ in range(2):                            # twice: plan state left by a solve must not matter
                shard.solve(rho_own, phi_own)
            torch.cuda.synchronize()
            out[r] = (lo, hi, phi_own)
            if eng is not None:
                eng.close()
        except Exception as e:                            # surfaced in the main thread
            errs.append((r, repr(e)))

    th = [threading.Thread(target=rank_main, args=(r,)) for r in range(world)]
    for t in th:
        t.start()
    for t in th:
        t.join(timeout=600)
    assert not errs, errs
    assert all(o is not None for o in out)
    phi = torch.empty_like(rho)
    for lo, hi, p in out:
        phi[lo:hi] = p
    return phi


@pytest.mark.parametrize("N,L,world", [(32, 5, 1), (32, 5, 2), (32, 5, 3), (32, 5, 5), (32, 3, 5), (16, 2, 2), (16, 1, 1), (16, 1, 2), (20, 4, 2), (64, 4, 3),
                                       (128, 4, 3), (256, 2, 2)])
def test_any_partition_of_the_levels_gives_the_bits_of_cm_potential(N, L, world):
    import paper_2301_06763_b200 as pkg
    pkg.build()
    dx0, G = 1.9 / N, 1.3
    rng = np.random.default_rng(1000 * N + 10 * L + world)
    rho = torch.from_numpy(rng.random((L, N, N, N)) + 0.1 * rng.standard_normal((L, N, N, N))).cuda()
    plan = pkg.Plan(N, L, dx0, G=G)
    ref = plan.potential(rho).clone()
    torch.cuda.synchronize()
    plan.close()
    got = _sharded(pkg, rho, N, L, dx0, G, world)
    assert torch.isfinite(got).all()
    assert torch.equal(got, ref), float((got - ref).abs().max() / ref.abs().max())


def test_shard_calls_reject_inconsistent_arguments():
    import paper_2301_06763_b200 as pkg
    pkg.build()
    N, L = 16, 3
    plan = pkg.Plan(N, L, 0.1)
    own = torch.zeros(L, N, N, N, dtype=torch.float64, device="cuda")
    small = torch.zeros((N // 2) ** 3, dtype=torch.float64, device="cuda")
    ring = torch.zeros((N // 2 + 2) ** 3, dtype=torch.float64, device="cuda")
    h, s = plan.handle, torch.cuda.current_stream().cuda_stream
    bad = [lambda: pkg.cm_shard_restrict(h, own.data_ptr(), 1, 1, None, None, s),                       # empty range
           lambda: pkg.cm_shard_restrict(h, own.data_ptr(), 0, 4, None, None, s),                       # beyond the nest
           lambda: pkg.cm_shard_restrict(h, own.data_ptr(), 0, 2, None, None, s),                       # hi < L needs rc_from_finer
           lambda: pkg.cm_shard_restrict(h, own.data_ptr(), 0, 3, small.data_ptr(), None, s),           # hi = L takes none
           lambda: pkg.cm_shard_restrict(h, own.data_ptr(), 1, 3, None, None, s),                       # lo > 0 needs rc_to_coarser
           lambda: pkg.cm_shard_forward(h, None, 0, 3, s),
           lambda: pkg.cm_shard_finish(h, own.data_ptr(), 1, 3, None, None, s),                         # lo > 0 needs the ring
           lambda: pkg.cm_shard_finish(h, own.data_ptr(), 0, 2, None, None, s),                         # hi < L must give one
           lambda: pkg.cm_shard_finish(h, own.data_ptr(), 0, 3, ring.data_ptr(), None, s)]
    for f in bad:
        with pytest.raises(pkg.CMError) as ei:
            f()
        assert ei.value.code == pkg.CM_EINVAL
    plan.close()
