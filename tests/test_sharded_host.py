"""Level sharding across ranks, host side, CPU: the partition of levels and the order of a rank's
steps and exchanges (`LevelShard`), run over gloo with a stand-in engine whose three steps have the same data
dependences as the solve (fine -> coarse chain, independent middle, coarse -> fine chain).  The arithmetic of the
stand-in is the test's own; the product's runs only on the GPU (tests/test_gpu_sharded.py)."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_is_contiguous_balanced_and_complete():
    from paper_2301_06763_b200.sharded import partition_levels
    for L in range(1, 14):
        for W in range(1, 11):
            parts = partition_levels(L, W)
            assert len(parts) == W and parts[0][0] == 0 and parts[-1][1] == L
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1 and sorted(sizes, reverse=True) == sizes
    assert partition_levels(10, 8) == [(0, 2), (2, 4), (4, 5), (5, 6), (6, 7), (7, 8), (8, 9), (9, 10)]
    assert partition_levels(2, 4) == [(0, 1), (1, 2), (2, 2), (2, 2)]
    with pytest.raises(ValueError):
        partition_levels(0, 2)


class _StandIn:
    """Three steps with the solve's dependences on scalar 'levels':
       rc[l] = rho[l+1] + rc[l+1] / 2 (rc[L-1] = 0);  w[l] = 3 rho[l] + rc[l];  h[l] = w[l] + h[l-1] / 4;  phi[l] = h[l]."""

    def __init__(self, torch, L, lo, hi):
        z = lambda: torch.zeros(1, dtype=torch.float64)
        self.L, self.rc, self.w = L, {}, {}
        self.rc_in = z() if hi < L else None
        self.rc_out = z() if lo > 0 else None
        self.ring_in = z() if lo > 0 else None
        self.ring_out = z() if hi < L else None
        self.calls = []

    def restrict(self, rho, lo, hi):
        self.calls.append("restrict")
        rc_next = float(self.rc_in) if hi < self.L else None
        for l in range(hi - 1, lo - 1, -1):
            self.rc[l] = 0.0 if l == self.L - 1 else (rc_next if l == hi - 1 else float(rho[l + 1 - lo]) + self.rc[l + 1] / 2)
        if lo > 0:
            self.rc_out[0] = float(rho[0]) + self.rc[lo] / 2

    def forward(self, rho, lo, hi):
        self.calls.append("forward")
        for l in range(lo, hi):
            self.w[l] = 3 * float(rho[l - lo]) + self.rc[l]

    def finish(self, phi, lo, hi):
        self.calls.append("finish")
        h = float(self.ring_in) if lo > 0 else 0.0
        for l in range(lo, hi):
            h = self.w[l] + h / 4
            phi[l - lo] = h
        if hi < self.L:
            self.ring_out[0] = h


def _expected(rho):
    L = len(rho)
    rc = [0.0] * L
    for l in range(L - 2, -1, -1):
        rc[l] = rho[l + 1] + rc[l + 1] / 2
    phi, h = [], 0.0
    for l in range(L):
        h = 3 * rho[l] + rc[l] + h / 4
        phi.append(h)
    return phi


def _rank_main(rank, world, port, L, out_dir):
    import json
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2301_06763_b200.sharded import LevelShard, partition_levels
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = partition_levels(L, world)[rank]
    eng = _StandIn(torch, L, lo, hi)
    log = []

    def send(t, peer):
        log.append(("send", peer))
        dist.send(t, peer)

    def recv(t, peer):
        log.append(("recv", peer))
        dist.recv(t, peer)

    shard = LevelShard(L, rank, world, eng, send, recv)
    rho_all = [1.0 + 0.37 * l * l for l in range(L)]
    rho_own = torch.tensor(rho_all[lo:hi], dtype=torch.float64)
    phi_own = torch.full((hi - lo,), float("nan"), dtype=torch.float64)
    for _ in range(2):                                  # two solves back to back: no message left over, no deadlock
        shard.solve(rho_own, phi_own)
    with open(os.path.join(out_dir, f"rank{rank}.json"), "w") as f:
        json.dump(dict(lo=lo, hi=hi, phi=phi_own.tolist(), log=log, calls=eng.calls), f)
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,L", [(2, 5), (3, 4), (3, 2)])
def test_level_shard_choreography_over_gloo(tmp_path, world, L):
    import json
    import torch.multiprocessing as mp
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    mp.spawn(_rank_main, args=(world, port, L, str(tmp_path)), nprocs=world, join=True)
    want = _expected([1.0 + 0.37 * l * l for l in range(L)])
    got = [None] * L
    for r in range(world):
        d = json.load(open(tmp_path / f"rank{r}.json"))
        for l in range(d["lo"], d["hi"]):
            got[l] = d["phi"][l - d["lo"]]
        active = d["hi"] > d["lo"]
        first, last = d["lo"] == 0, d["hi"] == L
        one = ([["recv", r + 1]] if active and not last else []) + ([["send", r - 1]] if active and not first else []) + \
              ([["recv", r - 1]] if active and not first else []) + ([["send", r + 1]] if active and not last else [])
        assert d["log"] == one * 2, (r, d["log"])
        assert d["calls"] == (["restrict", "forward", "finish"] * 2 if active else [])
    assert got == pytest.approx(want, rel=1e-15)
