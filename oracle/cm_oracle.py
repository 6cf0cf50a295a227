"""ctypes front end of the oracle (oracle/cm_oracle.c) + the Eq. 14 assembly.

ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).

The C file holds the primitives (restriction, Eq. 10 by brute force, the naive
(2N)^3 FFT convolution, the Eq. 3-6 prolongation); this file strings them
together in the paper's order:

    rhobar      = restriction cascade                       (L280-L282)
    Phi^l       = field(rhobar_l, full)                     (Eq. 10 on Omega^l)
    Phi^l_hole  = field(rhobar_l, cavity zeroed)            (L174-L176)
    ext_0 = 0;  ext_{l+1} = P[ext_l + Phi^l_hole]           (L176, reading 7: cascade)
    Phi(Omega^l) = Phi^l + ext_l                            (Eq. 14)

`method`: "direct" = literal O(N^6) sum, "fft" = the oracle's own padded FFT.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from functools import lru_cache

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cm_oracle.c")
_SO = os.path.join(_HERE, "libcm_oracle.so")

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
    return _SO


@lru_cache(maxsize=1)
def lib() -> C.CDLL:
    L = C.CDLL(build())
    L.orc_I0.restype = C.c_double
    L.orc_num_threads.restype = C.c_int
    L.orc_restrict.argtypes = [C.c_int, C.c_int, _dp, _dp]
    L.orc_field_direct.argtypes = [C.c_int, _dp, C.c_int, C.c_double, C.c_double, _dp]
    L.orc_field_direct_at.argtypes = [C.c_int, _dp, C.c_int, C.c_double, C.c_double, C.c_int, _ip, _dp]
    L.orc_green_hat.argtypes = [C.c_int, _dp]
    L.orc_field_fft.argtypes = [C.c_int, _dp, C.c_int, C.c_double, C.c_double, _dp, _dp, _dp]
    L.orc_prolong.argtypes = [C.c_int, _dp, _dp]
    L.orc_leaf_direct.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, _dp, C.c_int, _dp]
    L.orc_fft1d.argtypes = [C.c_long, _dp, C.c_int]
    L.orc_dft_naive.argtypes = [C.c_long, _dp, _dp, C.c_int, _dp, _dp]
    return L


def _p(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def _c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def I0() -> float:
    return float(lib().orc_I0())


def num_threads() -> int:
    return int(lib().orc_num_threads())


def restrict(rho: np.ndarray) -> np.ndarray:
    rho = _c(rho)
    L, N = rho.shape[0], rho.shape[1]
    out = np.empty_like(rho)
    lib().orc_restrict(N, L, _p(rho), _p(out))
    return out


def field_direct(rho_level: np.ndarray, hole: bool, G: float, dx: float) -> np.ndarray:
    r = _c(rho_level)
    N = r.shape[0]
    out = np.empty_like(r)
    lib().orc_field_direct(N, _p(r), int(hole), float(G), float(dx), _p(out))
    return out


def field_direct_at(rho_level: np.ndarray, hole: bool, G: float, dx: float, targets) -> np.ndarray:
    r = _c(rho_level)
    N = r.shape[0]
    t = np.ascontiguousarray(targets, dtype=np.int32).reshape(-1, 3)
    out = np.empty(t.shape[0])
    lib().orc_field_direct_at(N, _p(r), int(hole), float(G), float(dx), t.shape[0],
                              t.ctypes.data_as(_ip), _p(out))
    return out


def green_hat(N: int) -> np.ndarray:
    """FFT of the rearranged kernel on the doubled mesh, complex128 (2N,2N,2N)."""
    out = np.empty((2 * N, 2 * N, 2 * N), dtype=np.complex128)
    lib().orc_green_hat(N, out.ctypes.data_as(_dp))
    return out


def field_fft(rho_level: np.ndarray, hole: bool, G: float, dx: float, ghat: np.ndarray | None = None) -> np.ndarray:
    r = _c(rho_level)
    N = r.shape[0]
    if ghat is None:
        ghat = green_hat(N)
    assert ghat.dtype == np.complex128 and ghat.shape == (2 * N,) * 3 and ghat.flags.c_contiguous
    work = np.empty((2 * N,) * 3, dtype=np.complex128)
    out = np.empty_like(r)
    lib().orc_field_fft(N, _p(r), int(hole), float(G), float(dx), ghat.ctypes.data_as(_dp),
                        work.ctypes.data_as(_dp), _p(out))
    return out


def prolong(coarse: np.ndarray) -> np.ndarray:
    c = _c(coarse)
    out = np.empty_like(c)
    lib().orc_prolong(c.shape[0], _p(c), _p(out))
    return out


def leaf_direct(rho: np.ndarray, level: int, half0: float = 1.0, G: float = 1.0) -> np.ndarray:
    """Oracle-B: physical direct sum over leaf cells (bounds the METHOD's error)."""
    rho = _c(rho)
    L, N = rho.shape[0], rho.shape[1]
    out = np.empty((N, N, N))
    lib().orc_leaf_direct(N, L, float(half0), float(G), _p(rho), int(level), _p(out))
    return out


def fft1d(z: np.ndarray, sign: int) -> np.ndarray:
    a = np.ascontiguousarray(z, dtype=np.complex128).copy()
    lib().orc_fft1d(a.shape[0], a.ctypes.data_as(_dp), int(sign))
    return a


def dft_naive(z: np.ndarray, sign: int) -> np.ndarray:
    z = np.asarray(z, dtype=np.complex128)
    re, im = _c(z.real), _c(z.imag)
    ore, oim = np.empty_like(re), np.empty_like(im)
    lib().orc_dft_naive(z.shape[0], _p(re), _p(im), int(sign), _p(ore), _p(oim))
    return ore + 1j * oim


def solve(rho: np.ndarray, dx0: float, G: float = 1.0, method: str = "fft", return_parts: bool = False):
    """Whole method (Oracle-A): rho [L,N,N,N] -> Phi [L,N,N,N]."""
    rho = _c(rho)
    L, N = rho.shape[0], rho.shape[1]
    rhobar = restrict(rho)
    ghat = green_hat(N) if method == "fft" else None

    def field(l, hole):
        dx = dx0 / (1 << l)
        if method == "direct":
            return field_direct(rhobar[l], hole, G, dx)
        if method == "fft":
            return field_fft(rhobar[l], hole, G, dx, ghat)
        raise ValueError(method)

    phi = np.empty_like(rho)
    ext = np.zeros((N, N, N))
    parts = {"rhobar": rhobar, "full": [], "hole": [], "ext": []}
    for l in range(L):
        full = field(l, False)
        phi[l] = full + ext                                    # Eq. 14
        parts["full"].append(full)
        parts["ext"].append(ext)
        if l < L - 1:
            hole = field(l, True)
            parts["hole"].append(hole)
            ext = prolong(ext + hole)                          # tilde, cascaded
    return (phi, parts) if return_parts else phi


def solve_points(rho: np.ndarray, dx0: float, targets, G: float = 1.0) -> np.ndarray:
    """Phi at sampled cells [(level, k, j, i), ...] by direct sums only.

    The same definitions as solve(method="direct"), evaluated one output at a
    time so that full-size configs can be checked: Phi(l,t) = full_l(t) + ext_l(t),
    ext_0 = 0, ext_l(f) = 3/4 H_{l-1}(p) + 1/4 H_{l-1}(p+s), H_l = ext_l + hole_l.
    """
    rho = _c(rho)
    L, N = rho.shape[0], rho.shape[1]
    rhobar = restrict(rho)
    targets = [tuple(int(v) for v in t) for t in targets]

    # collect, level by level (fine -> coarse), the coarse cells whose H is needed
    needH = [set() for _ in range(L)]
    need_ext = [set() for _ in range(L)]
    for (l, k, j, i) in targets:
        need_ext[l].add((k, j, i))

    def parents(f):
        k, j, i = f
        p = (N // 4 + k // 2, N // 4 + j // 2, N // 4 + i // 2)
        s = (1 if k & 1 else -1, 1 if j & 1 else -1, 1 if i & 1 else -1)
        return p, (p[0] + s[0], p[1] + s[1], p[2] + s[2])

    for l in range(L - 1, 0, -1):
        for f in need_ext[l]:
            for c in parents(f):
                needH[l - 1].add(c)
                need_ext[l - 1].add(c)

    ext = [dict() for _ in range(L)]
    H = [dict() for _ in range(L)]
    for l in range(L):
        dx = dx0 / (1 << l)
        for f in need_ext[l]:
            if l == 0:
                ext[l][f] = 0.0
            else:
                p, q = parents(f)
                ext[l][f] = 0.75 * H[l - 1][p] + 0.25 * H[l - 1][q]
        cells = sorted(needH[l])
        if cells:
            hv = field_direct_at(rhobar[l], True, G, dx, np.array(cells, dtype=np.int32))
            for c, v in zip(cells, hv):
                H[l][c] = ext[l][c] + float(v)

    out = np.empty(len(targets))
    by_level = {}
    for n, (l, k, j, i) in enumerate(targets):
        by_level.setdefault(l, []).append((n, (k, j, i)))
    for l, items in by_level.items():
        dx = dx0 / (1 << l)
        fv = field_direct_at(rhobar[l], False, G, dx, np.array([c for _, c in items], dtype=np.int32))
        for (n, c), v in zip(items, fv):
            out[n] = float(v) + ext[l][c]
    return out
