"""ctypes binding of include/cm.h — argument marshalling only.

Every step of the path runs in libcm's CUDA kernels.  PyTorch supplies device memory
(`tensor.data_ptr()`) and streams (`torch.cuda.current_stream().cuda_stream`); nothing
here computes.  If libcm.so is missing or a call fails this raises — there is no
fallback of any kind.
"""
from __future__ import annotations

import ctypes as C
import os
from functools import lru_cache

from . import _build

CM_OK, CM_EINVAL, CM_ENOMEM, CM_ECUDA, CM_ENOTREADY = 0, -1, -2, -3, -4
CM_BUF_RESTRICTED, CM_BUF_HOLE, CM_BUF_KHAT = 0, 1, 2

EXPORTS = ["cm_plan_create", "cm_green_precompute", "cm_potential", "cm_potential_host", "cm_potential_profile",
           "cm_acceleration", "cm_potential_modified", "cm_potential_modified_triplets", "cm_plan_prepare_modified", "cm_direct_sum",
           "cm_plan_destroy",
           "cm_plan_set_G", "cm_plan_workspace_bytes", "cm_plan_kernel_launches", "cm_debug_copy",
           "cm_slot_to_freq", "cm_error_string", "cm_last_cuda_error",
           "cm_direct_sum_static", "cm_direct_sum_static_setup", "cm_static_last_error",
           "cm_shard_restrict", "cm_shard_forward", "cm_shard_finish"]
CM_STATIC_MAX_N = 32


class CMError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libcm error {code}: {msg}")
        self.code = code


@lru_cache(maxsize=1)
def lib() -> C.CDLL:
    if not os.path.exists(_build.SO):
        raise RuntimeError(f"{_build.SO} is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                           "(no CPU fallback exists)")
    L = C.CDLL(_build.SO)
    vp = C.c_void_p
    L.cm_plan_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_double, C.c_int]
    L.cm_green_precompute.argtypes = [vp]
    L.cm_potential.argtypes = [vp, vp, vp, vp]
    L.cm_potential_host.argtypes = [vp, vp, vp, vp]
    L.cm_potential_profile.argtypes = [vp, vp, vp, vp, C.POINTER(C.c_float), C.c_int]
    L.cm_acceleration.argtypes = [vp, vp, vp, vp]
    L.cm_potential_modified.argtypes = [vp, vp, vp, vp]
    L.cm_direct_sum.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp]
    L.cm_potential_modified_triplets.argtypes = [vp, vp, vp, C.c_int, vp]
    L.cm_plan_prepare_modified.argtypes = [vp, C.c_int, C.c_int]
    L.cm_plan_destroy.argtypes = [vp]
    L.cm_plan_set_G.argtypes = [vp, C.c_double]
    L.cm_plan_workspace_bytes.argtypes = [vp]
    L.cm_plan_workspace_bytes.restype = C.c_size_t
    L.cm_plan_kernel_launches.argtypes = [vp]
    L.cm_debug_copy.argtypes = [vp, C.c_int, vp, C.c_size_t, vp]
    L.cm_slot_to_freq.argtypes = [C.c_int, C.c_int]
    L.cm_error_string.argtypes = [C.c_int]
    L.cm_error_string.restype = C.c_char_p
    L.cm_last_cuda_error.argtypes = [vp]
    L.cm_last_cuda_error.restype = C.c_char_p
    L.cm_shard_restrict.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp, vp]
    L.cm_shard_forward.argtypes = [vp, vp, C.c_int, C.c_int, vp]
    L.cm_shard_finish.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp, vp]
    L.cm_direct_sum_static.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, vp, vp, vp]
    L.cm_direct_sum_static_setup.argtypes = []
    L.cm_static_last_error.argtypes = []
    L.cm_static_last_error.restype = C.c_char_p
    return L


def _check(code: int, plan=None):
    if code != CM_OK:
        msg = lib().cm_error_string(code).decode()
        if plan:
            extra = lib().cm_last_cuda_error(plan).decode()
            if extra:
                msg += " (" + extra + ")"
        raise CMError(code, msg)


# ---- the C ABI, name for name ------------------------------------------------------
def cm_plan_create(N: int, levels: int, dx0: float, refinement: int = 2) -> int:
    h = C.c_void_p()
    _check(lib().cm_plan_create(C.byref(h), int(N), int(levels), float(dx0), int(refinement)))
    return h.value


def cm_green_precompute(plan: int) -> None:
    _check(lib().cm_green_precompute(plan), plan)


def cm_potential(plan: int, rho_ptr: int, phi_ptr: int, stream: int = 0) -> None:
    _check(lib().cm_potential(plan, rho_ptr, phi_ptr, stream), plan)


def cm_potential_host(plan: int, rho_host_ptr: int, phi_host_ptr: int, stream: int = 0) -> None:
    _check(lib().cm_potential_host(plan, rho_host_ptr, phi_host_ptr, stream), plan)


def cm_potential_profile(plan: int, rho_ptr: int, phi_ptr: int, stream: int = 0) -> list:
    ms = (C.c_float * 7)()
    _check(lib().cm_potential_profile(plan, rho_ptr, phi_ptr, stream, ms, 7), plan)
    return [float(v) for v in ms]


def cm_potential_modified(plan: int, rho_ptr: int, phi_ptr: int, stream: int = 0) -> None:
    _check(lib().cm_potential_modified(plan, rho_ptr, phi_ptr, stream), plan)


def cm_potential_modified_triplets(plan: int, rho_ptr: int, phi_ptr: int, qdp_direct: int = 0, stream: int = 0) -> None:
    _check(lib().cm_potential_modified_triplets(plan, rho_ptr, phi_ptr, int(qdp_direct), stream), plan)


def cm_plan_prepare_modified(plan: int, depth: int, qdp_direct: int = 0) -> None:
    _check(lib().cm_plan_prepare_modified(plan, int(depth), int(qdp_direct)), plan)


def cm_direct_sum(plan: int, rho_ptr: int, src_level: int, dst_level: int, phi_ptr: int, stream: int = 0) -> None:
    _check(lib().cm_direct_sum(plan, rho_ptr, int(src_level), int(dst_level), phi_ptr, stream), plan)


def cm_shard_restrict(plan: int, rho_own_ptr: int, lo: int, hi: int, rc_from_finer_ptr, rc_to_coarser_ptr, stream: int = 0) -> None:
    _check(lib().cm_shard_restrict(plan, rho_own_ptr, int(lo), int(hi), rc_from_finer_ptr, rc_to_coarser_ptr, stream), plan)


def cm_shard_forward(plan: int, rho_own_ptr: int, lo: int, hi: int, stream: int = 0) -> None:
    _check(lib().cm_shard_forward(plan, rho_own_ptr, int(lo), int(hi), stream), plan)


def cm_shard_finish(plan: int, phi_own_ptr: int, lo: int, hi: int, ring_from_coarser_ptr, ring_to_finer_ptr, stream: int = 0) -> None:
    _check(lib().cm_shard_finish(plan, phi_own_ptr, int(lo), int(hi), ring_from_coarser_ptr, ring_to_finer_ptr, stream), plan)


def _check_static(code: int):
    if code != CM_OK:
        raise CMError(code, lib().cm_error_string(code).decode() + " (" + lib().cm_static_last_error().decode() + ")")


def cm_direct_sum_static(N: int, dx_src: float, dx_dst: float, G: float, rho_ptr: int, phi_ptr: int, stream: int = 0) -> None:
    _check_static(lib().cm_direct_sum_static(int(N), float(dx_src), float(dx_dst), float(G), rho_ptr, phi_ptr, stream))


def cm_direct_sum_static_setup() -> None:
    _check_static(lib().cm_direct_sum_static_setup())


def cm_static_last_error() -> str:
    return lib().cm_static_last_error().decode()


def cm_acceleration(plan: int, phi_ptr: int, g_ptr: int, stream: int = 0) -> None:
    _check(lib().cm_acceleration(plan, phi_ptr, g_ptr, stream), plan)


def cm_plan_destroy(plan: int) -> None:
    _check(lib().cm_plan_destroy(plan))


def cm_plan_set_G(plan: int, G: float) -> None:
    _check(lib().cm_plan_set_G(plan, float(G)), plan)


def cm_plan_workspace_bytes(plan: int) -> int:
    return int(lib().cm_plan_workspace_bytes(plan))


def cm_plan_kernel_launches(plan: int) -> int:
    return int(lib().cm_plan_kernel_launches(plan))


def cm_debug_copy(plan: int, which: int, dst_ptr: int, n_doubles: int, stream: int = 0) -> None:
    _check(lib().cm_debug_copy(plan, which, dst_ptr, n_doubles, stream), plan)


def cm_slot_to_freq(N: int, slot: int) -> int:
    return int(lib().cm_slot_to_freq(N, slot))


# ---- convenience wrappers over torch tensors (still marshalling only) --------------
def direct_sum_static(rho_src, dx_src: float, dx_dst: float, out, G: float = 1.0, stream=None):
    """Eq. B.7 without a plan and without any allocation (cm_direct_sum_static): rho_src and out are CUDA float64
    tensors [N, N, N] the caller owns, N <= CM_STATIC_MAX_N; out is overwritten and returned."""
    import torch
    N = int(rho_src.shape[0])
    for t in (rho_src, out):
        if t.dtype != torch.float64 or tuple(t.shape) != (N, N, N) or not t.is_contiguous() or t.device.type != "cuda":
            raise ValueError(f"expected contiguous float64 cuda tensors of shape {(N, N, N)}")
    s = torch.cuda.current_stream(rho_src.device).cuda_stream if stream is None else int(stream)
    with torch.cuda.device(rho_src.device):
        cm_direct_sum_static(N, dx_src, dx_dst, G, rho_src.data_ptr(), out.data_ptr(), s)
    return out


class Plan:
    """Owns a cm_plan; `potential` takes/returns CUDA float64 tensors [levels, N, N, N]."""

    def __init__(self, N: int, levels: int, dx0: float, G: float = 1.0, refinement: int = 2):
        self.N, self.levels, self.dx0 = int(N), int(levels), float(dx0)
        self._h = cm_plan_create(N, levels, dx0, refinement)
        if G != 1.0:
            cm_plan_set_G(self._h, G)
        cm_green_precompute(self._h)

    @property
    def handle(self) -> int:
        return self._h

    def _check_tensor(self, t, device_type):
        import torch
        shape = (self.levels, self.N, self.N, self.N)
        if t.dtype != torch.float64 or tuple(t.shape) != shape or not t.is_contiguous() or t.device.type != device_type:
            raise ValueError(f"expected contiguous float64 {device_type} tensor of shape {shape}")

    def potential(self, rho, phi=None, stream=None):
        import torch
        self._check_tensor(rho, "cuda")
        if phi is None:
            phi = torch.empty_like(rho)
        self._check_tensor(phi, "cuda")
        s = torch.cuda.current_stream(rho.device).cuda_stream if stream is None else int(stream)
        cm_potential(self._h, rho.data_ptr(), phi.data_ptr(), s)
        return phi

    def potential_modified(self, rho, phi=None, stream=None):
        """Modified (dipole) method over neighbouring pairs, Eq. B.1-B.2 (cm_potential_modified)."""
        import torch
        self._check_tensor(rho, "cuda")
        if phi is None:
            phi = torch.empty_like(rho)
        self._check_tensor(phi, "cuda")
        s = torch.cuda.current_stream(rho.device).cuda_stream if stream is None else int(stream)
        cm_potential_modified(self._h, rho.data_ptr(), phi.data_ptr(), s)
        return phi

    def potential_modified_triplets(self, rho, phi=None, qdp_direct: bool = False, stream=None):
        """Modified method over three neighbouring grids, Eq. B.3-B.6 (cm_potential_modified_triplets)."""
        import torch
        self._check_tensor(rho, "cuda")
        if phi is None:
            phi = torch.empty_like(rho)
        self._check_tensor(phi, "cuda")
        s = torch.cuda.current_stream(rho.device).cuda_stream if stream is None else int(stream)
        cm_potential_modified_triplets(self._h, rho.data_ptr(), phi.data_ptr(), int(bool(qdp_direct)), s)
        return phi

    def prepare_modified(self, depth: int = 2, qdp_direct: bool = False):
        """Allocate the expanded-grid plans of the modified method up front (cm_plan_prepare_modified)."""
        cm_plan_prepare_modified(self._h, depth, int(bool(qdp_direct)))

    def direct_sum(self, rho, src_level: int, dst_level: int, stream=None):
        """Eq. B.7: potential of level src_level's mass on the cells of level dst_level, [N, N, N]."""
        import torch
        self._check_tensor(rho, "cuda")
        out = torch.empty((self.N, self.N, self.N), dtype=torch.float64, device=rho.device)
        s = torch.cuda.current_stream(rho.device).cuda_stream if stream is None else int(stream)
        cm_direct_sum(self._h, rho.data_ptr(), src_level, dst_level, out.data_ptr(), s)
        return out

    def acceleration(self, phi, g=None, stream=None):
        """g[levels, 3, N, N, N] = -grad phi (cm_acceleration)."""
        import torch
        self._check_tensor(phi, "cuda")
        shape = (self.levels, 3, self.N, self.N, self.N)
        if g is None:
            g = torch.empty(shape, dtype=torch.float64, device=phi.device)
        if g.dtype != torch.float64 or tuple(g.shape) != shape or not g.is_contiguous() or g.device.type != "cuda":
            raise ValueError(f"expected contiguous float64 cuda tensor of shape {shape}")
        s = torch.cuda.current_stream(phi.device).cuda_stream if stream is None else int(stream)
        cm_acceleration(self._h, phi.data_ptr(), g.data_ptr(), s)
        return g

    def potential_host(self, rho_host, phi_host=None, stream=None):
        import torch
        self._check_tensor(rho_host, "cpu")
        if phi_host is None:
            phi_host = torch.empty_like(rho_host).pin_memory()
        self._check_tensor(phi_host, "cpu")
        s = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
        cm_potential_host(self._h, rho_host.data_ptr(), phi_host.data_ptr(), s)
        return phi_host

    def potential_profile(self, rho, phi, stream=None) -> dict:
        import torch
        self._check_tensor(rho, "cuda")
        self._check_tensor(phi, "cuda")
        s = torch.cuda.current_stream(rho.device).cuda_stream if stream is None else int(stream)
        ms = cm_potential_profile(self._h, rho.data_ptr(), phi.data_ptr(), s)
        return dict(zip(["restrict", "P1_x_fwd", "P2_y_fwd", "P3_z_conv", "P4_y_inv", "P5_x_inv", "prolong_sum"], ms))

    def debug_buffer(self, which: int):
        import torch
        N, L = self.N, self.levels
        shape = {CM_BUF_RESTRICTED: (max(L - 1, 0), N // 2, N // 2, N // 2), CM_BUF_HOLE: (L, N, N, N),
                 CM_BUF_KHAT: (2 * N, 2 * N, 2 * N)}[which]
        out = torch.empty(shape, dtype=torch.float64, device="cuda")
        if out.numel():
            cm_debug_copy(self._h, which, out.data_ptr(), out.numel(), torch.cuda.current_stream().cuda_stream)
        return out

    @property
    def workspace_bytes(self) -> int:
        return cm_plan_workspace_bytes(self._h)

    @property
    def kernel_launches(self) -> int:
        return cm_plan_kernel_launches(self._h)

    def close(self):
        if getattr(self, "_h", None):
            cm_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
