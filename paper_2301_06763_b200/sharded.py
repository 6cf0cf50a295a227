"""The solve sharded by levels across GPUs (the fields of different grids are independent).

One process per GPU; rank r owns the contiguous levels [lo, hi) given by `partition_levels` and holds only their
densities and potentials.  A solve is libcm's three shard calls (include/cm.h) with two small neighbour exchanges:

    fine -> coarse   (N/2)^3 fp64 per rank boundary: the projected density of the next rank's coarsest level
    P1..P4           85-90 % of the work, no exchange
    coarse -> fine   (N/2+2)^3 fp64 per rank boundary: ext + Phi_hole of the previous rank's finest level

Here is only the choreography — who waits for whom — and the marshalling; every step of the arithmetic runs in libcm's
kernels.  `LevelShard` takes the three steps as an `engine` and the transport as two callables, so that the ordering can
be exercised over gloo on CPU (tests/test_host_logic.py) and the data path on one GPU, rank after rank
(tests/test_gpu_sharded.py); `ShardedSolver` wires it to libcm and torch.distributed (NCCL).
"""
from __future__ import annotations

from . import binding as _b


def partition_levels(levels: int, world: int):
    """Contiguous level ranges, one per rank, sizes differing by at most one (the first levels % world ranks take the
    extra level); ranks beyond `levels` get an empty range (lo == hi == levels) and take no part."""
    if levels < 1 or world < 1:
        raise ValueError("levels and world must be positive")
    base, extra = divmod(levels, world)
    out, lo = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((lo, lo + n))
        lo += n
    return out


class LevelShard:
    """The order of one rank's steps in a level-sharded solve.

    engine: restrict(rho_own, lo, hi), forward(rho_own, lo, hi), finish(phi_own, lo, hi) and the four exchange
    buffers rc_in / rc_out / ring_in / ring_out (None where the rank has no such neighbour);
    send(buffer, peer_rank) / recv(buffer, peer_rank): blocking or stream-ordered point-to-point transport.
    """

    def __init__(self, levels: int, rank: int, world: int, engine, send, recv):
        parts = partition_levels(levels, world)
        self.levels, self.rank, self.world = levels, rank, world
        self.lo, self.hi = parts[rank]
        self.active = self.hi > self.lo
        # neighbours in the chain: ranges are contiguous and the empty ones come last
        self.prev = rank - 1 if self.active and self.lo > 0 else None
        self.next = rank + 1 if self.active and self.hi < levels else None
        self.engine, self._send, self._recv = engine, send, recv

    def solve(self, rho_own, phi_own):
        if not self.active:
            return phi_own
        e, lo, hi = self.engine, self.lo, self.hi
        if self.next is not None:
            self._recv(e.rc_in, self.next)           # projection of level hi onto the cavity of level hi - 1
        e.restrict(rho_own, lo, hi)
        if self.prev is not None:
            self._send(e.rc_out, self.prev)          # leaves before the passes start: the chain does not wait for them
        e.forward(rho_own, lo, hi)
        if self.prev is not None:
            self._recv(e.ring_in, self.prev)         # ext + Phi_hole of level lo - 1 on its cavity grown by one cell
        e.finish(phi_own, lo, hi)
        if self.next is not None:
            self._send(e.ring_out, self.next)
        return phi_own


class LibcmEngine:
    """The three shard calls of include/cm.h on a plan of the whole nest, plus the exchange buffers (CUDA tensors)."""

    def __init__(self, N: int, levels: int, dx0: float, lo: int, hi: int, G: float = 1.0, device=None):
        import torch
        self.N, self.levels, self.lo, self.hi = int(N), int(levels), int(lo), int(hi)
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        with torch.cuda.device(self.device):
            self.plan = _b.Plan(N, levels, dx0, G=G)
        H, B = N // 2, N // 2 + 2
        mk = lambda n: torch.empty(n, dtype=torch.float64, device=self.device)
        self.rc_in = mk(H ** 3) if hi < levels else None
        self.rc_out = mk(H ** 3) if lo > 0 else None
        self.ring_in = mk(B ** 3) if lo > 0 else None
        self.ring_out = mk(B ** 3) if hi < levels else None

    def _stream(self):
        import torch
        return torch.cuda.current_stream(self.device).cuda_stream

    @staticmethod
    def _ptr(t):
        return None if t is None else t.data_ptr()

    def check(self, t):
        import torch
        shape = (self.hi - self.lo, self.N, self.N, self.N)
        if t.dtype != torch.float64 or tuple(t.shape) != shape or not t.is_contiguous() or t.device != self.device:
            raise ValueError(f"expected contiguous float64 tensor of shape {shape} on {self.device}")

    def restrict(self, rho_own, lo, hi):
        self.check(rho_own)
        _b.cm_shard_restrict(self.plan.handle, rho_own.data_ptr(), lo, hi, self._ptr(self.rc_in), self._ptr(self.rc_out), self._stream())

    def forward(self, rho_own, lo, hi):
        _b.cm_shard_forward(self.plan.handle, rho_own.data_ptr(), lo, hi, self._stream())

    def finish(self, phi_own, lo, hi):
        self.check(phi_own)
        _b.cm_shard_finish(self.plan.handle, phi_own.data_ptr(), lo, hi, self._ptr(self.ring_in), self._ptr(self.ring_out), self._stream())

    def close(self):
        self.plan.close()


class ShardedSolver:
    """Level-sharded solve over a torch.distributed process group (NCCL): rank r of `group` solves its levels.

        solver = ShardedSolver(N, levels, dx0)            # after init_process_group("nccl") and torch.cuda.set_device
        phi_own = solver.solve(rho_own)                   # [hi - lo, N, N, N] float64 CUDA tensors, levels solver.lo .. solver.hi - 1
    """

    def __init__(self, N: int, levels: int, dx0: float, G: float = 1.0, group=None):
        import torch.distributed as dist
        self._dist, self._group = dist, group
        rank, world = dist.get_rank(group), dist.get_world_size(group)
        lo, hi = partition_levels(levels, world)[rank]
        self.engine = LibcmEngine(N, levels, dx0, lo, hi, G=G) if hi > lo else None
        self.shard = LevelShard(levels, rank, world, self.engine, self._send, self._recv)
        self.lo, self.hi, self.N = lo, hi, int(N)

    def _peer(self, r):
        return r if self._group is None else self._dist.get_global_rank(self._group, r)

    def _send(self, t, peer):
        self._dist.send(t, self._peer(peer), group=self._group)

    def _recv(self, t, peer):
        self._dist.recv(t, self._peer(peer), group=self._group)

    def solve(self, rho_own, phi_own=None):
        import torch
        if self.engine is None:
            return phi_own
        if phi_own is None:
            phi_own = torch.empty_like(rho_own)
        return self.shard.solve(rho_own, phi_own)

    def close(self):
        if self.engine is not None:
            self.engine.close()
