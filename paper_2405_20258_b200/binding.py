"""ctypes binding with the same names as the C-ABI entry points of include/rpa_b200.h.

Tensors are torch CUDA tensors (complex128 / float64, contiguous); the binding passes their data pointers and the
current torch CUDA stream.  There is no fallback: if the shared library is missing or no CUDA device is present the
calls raise."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

EXPORTED_SYMBOLS = [
    "rpa_create", "rpa_destroy", "rpa_last_error", "rpa_workspace_bytes", "rpa_energy_workspace_bytes",
    "rpa_set_workspace", "rpa_mtxel", "rpa_chi0_static", "rpa_subspace_basis", "rpa_chi_subspace_freq",
    "rpa_correlation_energy", "rpa_energy_device", "rpa_energy_host", "rpa_fp64_peak", "rpa_launch_count",
    "rpa_profile_begin", "rpa_profile_end", "rpa_chi0_static_occ", "rpa_chi_subspace_freq_occ",
    "rpa_epsilon_inverse", "rpa_epsilon_inverse_workspace_bytes", "rpa_basis_info", "rpa_basis_quality",
    "rpa_pass_begin", "rpa_pass1_chi0", "rpa_pass_basis", "rpa_pass2_chis", "rpa_pass_energy", "rpa_pass_end",
    "rpa_noalloc_max_pairs", "rpa_noalloc_setup", "rpa_chi0_static_noalloc",
]


class RpaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"rpa error {code}: {msg}")
        self.code = code


def library_path() -> str:
    return os.path.join(_HERE, "librpa_b200.so")


def load_library(build_if_missing: bool = True):
    """dlopen librpa_b200.so (building it in-tree with nvcc first if it is missing or stale)."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    if build_if_missing:
        from . import _build
        try:
            _build.build()
        except FileNotFoundError:       # no nvcc on this machine: an existing library is used as it is
            if not os.path.exists(path):
                raise
        # any other failure (a compile error after a source edit) propagates: never run a stale binary silently
    if not os.path.exists(path):
        raise RpaError(-3, f"{path} is missing: build it with `python -m paper_2405_20258_b200._build` (no CPU fallback)")
    lib = C.CDLL(path)
    vp, ci, cd, pd, pi = C.c_void_p, C.c_int, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_int)
    lib.rpa_create.argtypes = [C.POINTER(vp), pd, pi, ci, C.POINTER(C.c_int32), pd, ci, C.POINTER(C.c_int32), ci, vp]
    lib.rpa_create.restype = ci
    lib.rpa_destroy.argtypes = [vp]
    lib.rpa_destroy.restype = ci
    lib.rpa_last_error.argtypes = [vp]
    lib.rpa_last_error.restype = C.c_char_p
    lib.rpa_workspace_bytes.argtypes = [vp, ci, ci, ci, ci]
    lib.rpa_workspace_bytes.restype = C.c_size_t
    lib.rpa_energy_workspace_bytes.argtypes = [vp, ci, ci, ci, ci, ci]
    lib.rpa_energy_workspace_bytes.restype = C.c_size_t
    lib.rpa_set_workspace.argtypes = [vp, vp, C.c_size_t]
    lib.rpa_set_workspace.restype = ci
    lib.rpa_mtxel.argtypes = [vp, vp, ci, vp, ci, vp]
    lib.rpa_mtxel.restype = ci
    lib.rpa_chi0_static.argtypes = [vp, vp, ci, ci, vp, vp, ci, vp]
    lib.rpa_chi0_static.restype = ci
    lib.rpa_subspace_basis.argtypes = [vp, vp, ci, cd, vp, vp, pi]
    lib.rpa_subspace_basis.restype = ci
    lib.rpa_chi_subspace_freq.argtypes = [vp, vp, ci, ci, vp, vp, vp, ci, vp, ci, ci, vp]
    lib.rpa_chi_subspace_freq.restype = ci
    lib.rpa_chi0_static_occ.argtypes = [vp, vp, ci, ci, vp, vp, vp, vp, ci, vp]
    lib.rpa_chi0_static_occ.restype = ci
    lib.rpa_chi_subspace_freq_occ.argtypes = [vp, vp, ci, ci, vp, vp, vp, vp, vp, ci, vp, ci, ci, vp]
    lib.rpa_chi_subspace_freq_occ.restype = ci
    lib.rpa_epsilon_inverse.argtypes = [vp, vp, ci, ci, vp]
    lib.rpa_epsilon_inverse.restype = ci
    lib.rpa_epsilon_inverse_workspace_bytes.argtypes = [vp, ci, ci]
    lib.rpa_epsilon_inverse_workspace_bytes.restype = C.c_size_t
    lib.rpa_correlation_energy.argtypes = [vp, vp, ci, vp, ci, pd, pd]
    lib.rpa_correlation_energy.restype = ci
    energy_args = [vp, vp, ci, vp, ci, vp, vp, ci, ci, cd, vp, vp, ci, ci, pd, pd, pd, pd]
    lib.rpa_energy_device.argtypes = energy_args
    lib.rpa_energy_device.restype = ci
    lib.rpa_energy_host.argtypes = energy_args
    lib.rpa_energy_host.restype = ci
    lib.rpa_pass_begin.argtypes = [vp, vp, ci, vp, ci, vp, vp, ci, ci, vp, ci, ci, ci]
    lib.rpa_pass_begin.restype = ci
    lib.rpa_pass1_chi0.argtypes = [vp, C.POINTER(vp)]
    lib.rpa_pass1_chi0.restype = ci
    lib.rpa_pass_basis.argtypes = [vp, cd, ci, C.POINTER(vp), C.POINTER(vp)]
    lib.rpa_pass_basis.restype = ci
    lib.rpa_pass2_chis.argtypes = [vp, C.POINTER(vp)]
    lib.rpa_pass2_chis.restype = ci
    lib.rpa_pass_energy.argtypes = [vp, vp, pd, pd, pd, pd]
    lib.rpa_pass_energy.restype = ci
    lib.rpa_pass_end.argtypes = [vp]
    lib.rpa_pass_end.restype = ci
    lib.rpa_noalloc_max_pairs.argtypes = []
    lib.rpa_noalloc_max_pairs.restype = C.c_longlong
    lib.rpa_noalloc_setup.argtypes = [vp]
    lib.rpa_noalloc_setup.restype = ci
    lib.rpa_chi0_static_noalloc.argtypes = [vp, vp, ci, ci, vp, vp, ci, vp]
    lib.rpa_chi0_static_noalloc.restype = ci
    lib.rpa_fp64_peak.argtypes = [vp, ci, ci, pd]
    lib.rpa_fp64_peak.restype = ci
    lib.rpa_profile_begin.argtypes = [vp]
    lib.rpa_profile_begin.restype = ci
    lib.rpa_profile_end.argtypes = [vp, pd, C.POINTER(C.c_longlong)]
    lib.rpa_profile_end.restype = ci
    lib.rpa_basis_info.argtypes = [vp, pi, pi, pi]
    lib.rpa_basis_info.restype = ci
    lib.rpa_basis_quality.argtypes = [vp, pd, pd]
    lib.rpa_basis_quality.restype = ci
    lib.rpa_launch_count.argtypes = [vp]
    lib.rpa_launch_count.restype = C.c_longlong
    _LIB = lib
    return lib


def _check(ctx, rc):
    if rc != 0:
        msg = load_library().rpa_last_error(ctx)
        raise RpaError(rc, msg.decode() if msg else "?")


def _dev(t, dtype=None):
    """device pointer of a contiguous CUDA tensor"""
    import torch
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda or not t.is_contiguous():
        raise TypeError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _shape(name, t, *dims):
    """The C ABI receives raw pointers, so a mis-shaped tensor would be an out-of-bounds device access with no error:
    every array is checked against the sizes the call passes to the library before the call is made."""
    got = tuple(int(x) for x in t.shape)
    if got != tuple(int(d) for d in dims):
        raise TypeError(f"{name}: expected shape {tuple(int(d) for d in dims)}, got {got}")


class RpaContext:
    """Owns an rpa_ctx* and the workspace tensor lent to it."""

    def __init__(self, handle, device, n_g=None, n_pw=None):
        self.handle = handle
        self.device = device
        self.workspace = None
        self.n_g, self.n_pw = n_g, n_pw
        self._pass = None

    def close(self):
        if self.handle:
            load_library().rpa_destroy(self.handle)
            self.handle = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def rpa_create(cell, fft, g_eps, vcoul, g_wfn, device: int = 0, stream=None) -> RpaContext:
    import torch
    lib = load_library()
    if not torch.cuda.is_available():
        raise RpaError(-3, "no CUDA device: the RPA hot path has no CPU fallback")
    cell = np.ascontiguousarray(cell, dtype=np.float64).reshape(9)
    fft = np.ascontiguousarray(fft, dtype=np.int32).reshape(3)
    g_eps = np.ascontiguousarray(g_eps, dtype=np.int32)
    g_wfn = np.ascontiguousarray(g_wfn, dtype=np.int32)
    vcoul = np.ascontiguousarray(vcoul, dtype=np.float64)
    if stream is None:
        stream = torch.cuda.current_stream(device).cuda_stream
    h = C.c_void_p()
    rc = lib.rpa_create(C.byref(h), cell.ctypes.data_as(C.POINTER(C.c_double)), fft.ctypes.data_as(C.POINTER(C.c_int)),
                        g_eps.shape[0], g_eps.ctypes.data_as(C.POINTER(C.c_int32)),
                        vcoul.ctypes.data_as(C.POINTER(C.c_double)), g_wfn.shape[0],
                        g_wfn.ctypes.data_as(C.POINTER(C.c_int32)), device, C.c_void_p(stream))
    _check(None, rc)
    return RpaContext(h, device, n_g=int(g_eps.shape[0]), n_pw=int(g_wfn.shape[0]))


def rpa_destroy(ctx: RpaContext):
    ctx.close()


def rpa_workspace_bytes(ctx, nvb, nc, n_eig, n_w) -> int:
    return int(load_library().rpa_workspace_bytes(ctx.handle, nvb, nc, n_eig, n_w))


def rpa_energy_workspace_bytes(ctx, nv, nc, nvb, n_eig, n_w) -> int:
    return int(load_library().rpa_energy_workspace_bytes(ctx.handle, nv, nc, nvb, n_eig, n_w))


def rpa_set_workspace(ctx, tensor):
    """Lend a torch uint8 CUDA tensor as scratch memory (kept alive by the context)."""
    ptr = _dev(tensor)
    _check(ctx.handle, load_library().rpa_set_workspace(ctx.handle, ptr, tensor.numel() * tensor.element_size()))
    ctx.workspace = tensor


def rpa_mtxel(ctx, psi_v, psi_c, M):
    import torch
    nvb, nc = psi_v.shape[0], psi_c.shape[0]
    _shape("psi_v", psi_v, nvb, ctx.n_pw)
    _shape("psi_c", psi_c, nc, ctx.n_pw)
    _shape("M", M, nvb, nc, ctx.n_g)
    _check(ctx.handle, load_library().rpa_mtxel(ctx.handle, _dev(psi_v, torch.complex128), nvb,
                                                _dev(psi_c, torch.complex128), nc, _dev(M, torch.complex128)))
    return M


def _pair_shapes(ctx, M, e_v, e_c, f_v=None, f_c=None):
    nvb, nc = e_v.shape[0], e_c.shape[0]
    _shape("e_v", e_v, nvb)
    _shape("e_c", e_c, nc)
    _shape("M", M, nvb, nc, ctx.n_g)
    if f_v is not None:
        _shape("f_v", f_v, nvb)
        _shape("f_c", f_c, nc)


def _freq_shapes(ctx, Cmat, n_eig, omega, chi_s):
    if Cmat is not None:
        _shape("C", Cmat, n_eig, ctx.n_g)
    elif n_eig != ctx.n_g:
        raise TypeError(f"C is None (full basis): n_eig must be n_g = {ctx.n_g}, got {n_eig}")
    _shape("omega", omega, omega.shape[0])
    _shape("chi_s", chi_s, omega.shape[0], n_eig, n_eig)


def rpa_chi0_static(ctx, M, e_v, e_c, accumulate, chi0):
    import torch
    _pair_shapes(ctx, M, e_v, e_c)
    _shape("chi0", chi0, ctx.n_g, ctx.n_g)
    _check(ctx.handle, load_library().rpa_chi0_static(ctx.handle, _dev(M, torch.complex128), e_v.shape[0], e_c.shape[0],
                                                      _dev(e_v, torch.float64), _dev(e_c, torch.float64),
                                                      int(bool(accumulate)), _dev(chi0, torch.complex128)))
    return chi0


def rpa_noalloc_max_pairs() -> int:
    return int(load_library().rpa_noalloc_max_pairs())


def rpa_noalloc_setup(ctx):
    _check(ctx.handle, load_library().rpa_noalloc_setup(ctx.handle))


def rpa_chi0_static_noalloc(ctx, M, e_v, e_c, accumulate, chi0):
    """rpa_chi0_static with its scratch in a device array built into the library (no workspace, no allocation); at most
    rpa_noalloc_max_pairs() pairs per call; calls that overlap on the GPU race on that array."""
    import torch
    _pair_shapes(ctx, M, e_v, e_c)
    _shape("chi0", chi0, ctx.n_g, ctx.n_g)
    _check(ctx.handle, load_library().rpa_chi0_static_noalloc(ctx.handle, _dev(M, torch.complex128), e_v.shape[0], e_c.shape[0],
                                                              _dev(e_v, torch.float64), _dev(e_c, torch.float64),
                                                              int(bool(accumulate)), _dev(chi0, torch.complex128)))
    return chi0


def rpa_subspace_basis(ctx, chi0, n_eig, tol, Cmat, lam):
    import torch
    _shape("chi0", chi0, ctx.n_g, ctx.n_g)
    _shape("C", Cmat, n_eig, ctx.n_g)
    _shape("lambda", lam, n_eig)
    iters = C.c_int(0)
    _check(ctx.handle, load_library().rpa_subspace_basis(ctx.handle, _dev(chi0, torch.complex128), n_eig, float(tol),
                                                         _dev(Cmat, torch.complex128), _dev(lam, torch.float64),
                                                         C.byref(iters)))
    return iters.value


def rpa_chi_subspace_freq(ctx, M, e_v, e_c, Cmat, n_eig, omega, accumulate, chi_s):
    import torch
    _pair_shapes(ctx, M, e_v, e_c)
    _freq_shapes(ctx, Cmat, n_eig, omega, chi_s)
    _check(ctx.handle, load_library().rpa_chi_subspace_freq(
        ctx.handle, _dev(M, torch.complex128), e_v.shape[0], e_c.shape[0], _dev(e_v, torch.float64),
        _dev(e_c, torch.float64), _dev(Cmat, torch.complex128) if Cmat is not None else None, n_eig,
        _dev(omega, torch.float64), omega.shape[0], int(bool(accumulate)), _dev(chi_s, torch.complex128)))
    return chi_s


def rpa_chi0_static_occ(ctx, M, e_v, e_c, f_v, f_c, accumulate, chi0):
    import torch
    f64, c128 = torch.float64, torch.complex128
    _pair_shapes(ctx, M, e_v, e_c, f_v, f_c)
    _shape("chi0", chi0, ctx.n_g, ctx.n_g)
    _check(ctx.handle, load_library().rpa_chi0_static_occ(ctx.handle, _dev(M, c128), e_v.shape[0], e_c.shape[0], _dev(e_v, f64),
                                                          _dev(e_c, f64), _dev(f_v, f64), _dev(f_c, f64), int(bool(accumulate)),
                                                          _dev(chi0, c128)))
    return chi0


def rpa_chi_subspace_freq_occ(ctx, M, e_v, e_c, f_v, f_c, Cmat, n_eig, omega, accumulate, chi_s):
    import torch
    f64, c128 = torch.float64, torch.complex128
    _pair_shapes(ctx, M, e_v, e_c, f_v, f_c)
    _freq_shapes(ctx, Cmat, n_eig, omega, chi_s)
    _check(ctx.handle, load_library().rpa_chi_subspace_freq_occ(
        ctx.handle, _dev(M, c128), e_v.shape[0], e_c.shape[0], _dev(e_v, f64), _dev(e_c, f64), _dev(f_v, f64), _dev(f_c, f64),
        _dev(Cmat, c128) if Cmat is not None else None, n_eig, _dev(omega, f64), omega.shape[0], int(bool(accumulate)),
        _dev(chi_s, c128)))
    return chi_s


def rpa_epsilon_inverse_workspace_bytes(ctx, n_eig, n_w) -> int:
    return int(load_library().rpa_epsilon_inverse_workspace_bytes(ctx.handle, n_eig, n_w))


def rpa_epsilon_inverse(ctx, chi_s, eps_inv):
    import torch
    n_w, n_eig = chi_s.shape[0], chi_s.shape[1]
    _shape("chi_s", chi_s, n_w, n_eig, n_eig)
    _shape("eps_inv", eps_inv, n_w, n_eig, n_eig)
    _check(ctx.handle, load_library().rpa_epsilon_inverse(ctx.handle, _dev(chi_s, torch.complex128), n_eig, n_w,
                                                          _dev(eps_inv, torch.complex128)))
    return eps_inv


def rpa_correlation_energy(ctx, chi_s, n_eig, weight):
    import torch
    n_w = weight.shape[0]
    _shape("weight", weight, n_w)
    _shape("chi_s", chi_s, n_w, n_eig, n_eig)
    e = C.c_double(0.0)
    per = (C.c_double * n_w)()
    _check(ctx.handle, load_library().rpa_correlation_energy(ctx.handle, _dev(chi_s, torch.complex128), n_eig,
                                                             _dev(weight, torch.float64), n_w, C.byref(e), per))
    return e.value, np.array(per[:])


def _energy(fn_name, ctx, psi_v, psi_c, e_v, e_c, nvb, n_eig, tol, omega, weight, keep_m, ptr):
    nv, nc, n_w = psi_v.shape[0], psi_c.shape[0], omega.shape[0]
    _shape("psi_v", psi_v, nv, ctx.n_pw)
    _shape("psi_c", psi_c, nc, ctx.n_pw)
    _shape("e_v", e_v, nv)
    _shape("e_c", e_c, nc)
    _shape("weight", weight, n_w)
    if not (1 <= int(n_eig) <= ctx.n_g):
        raise TypeError(f"n_eig = {n_eig} not in 1..n_g = {ctx.n_g}")
    e = C.c_double(0.0)
    lam = (C.c_double * n_eig)()
    per = (C.c_double * n_w)()
    ms = (C.c_double * 5)()
    fn = getattr(load_library(), fn_name)
    _check(ctx.handle, fn(ctx.handle, ptr(psi_v), nv, ptr(psi_c), nc, ptr(e_v), ptr(e_c), int(nvb), int(n_eig), float(tol),
                          ptr(omega), ptr(weight), n_w, int(bool(keep_m)), C.byref(e), lam, per, ms))
    return dict(E_c=e.value, lam=np.array(lam[:]), t=np.array(per[:]),
                stage_ms=dict(zip(("mtxel", "chi0_static", "basis", "chi_freq", "energy"), ms[:])))


def rpa_energy_device(ctx, psi_v, psi_c, e_v, e_c, nvb, n_eig, tol, omega, weight, keep_m=False):
    """All inputs are CUDA tensors."""
    return _energy("rpa_energy_device", ctx, psi_v, psi_c, e_v, e_c, nvb, n_eig, tol, omega, weight, keep_m, _dev)


def rpa_energy_host(ctx, psi_v, psi_c, e_v, e_c, nvb, n_eig, tol, omega, weight, keep_m=False):
    """All inputs are HOST arrays (numpy, or CPU torch tensors, ideally pinned); copies happen inside the call."""
    import torch

    def hptr(a):
        if isinstance(a, torch.Tensor):
            if a.is_cuda or not a.is_contiguous():
                raise TypeError("expected a contiguous CPU tensor")
            return C.c_void_p(a.data_ptr())
        if not isinstance(a, np.ndarray) or not a.flags["C_CONTIGUOUS"]:
            raise TypeError("expected a C-contiguous numpy array")
        return C.c_void_p(a.ctypes.data)

    return _energy("rpa_energy_host", ctx, psi_v, psi_c, e_v, e_c, nvb, n_eig, tol, omega, weight, keep_m, hptr)


def _ws_view(ctx, ptr, dtype, *shape):
    """A torch view (no copy) of an array the library placed inside the workspace tensor the context was lent."""
    import torch
    ws = ctx.workspace
    if ws is None or ptr is None:
        raise RpaError(-2, "no workspace tensor is lent to the context")
    n = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
    off = int(ptr) - ws.data_ptr()
    if off < 0 or off + n > ws.numel() * ws.element_size():
        raise RpaError(-2, "pointer returned by the library lies outside the workspace tensor")
    return ws[off:off + n].view(dtype).view(*shape)


def rpa_pass_begin(ctx, psi_v, psi_c, e_v, e_c, nvb, n_eig, omega, keep_m=True, timing=True):
    """Opens the pass-level sequence (rpa_b200.h): all inputs are CUDA tensors, kept alive by the context until rpa_pass_end."""
    import torch
    nv, nc, n_w = psi_v.shape[0], psi_c.shape[0], omega.shape[0]
    _shape("psi_v", psi_v, nv, ctx.n_pw)
    _shape("psi_c", psi_c, nc, ctx.n_pw)
    _shape("e_v", e_v, nv)
    _shape("e_c", e_c, nc)
    if not (1 <= int(n_eig) <= ctx.n_g):
        raise TypeError(f"n_eig = {n_eig} not in 1..n_g = {ctx.n_g}")
    c128, f64 = torch.complex128, torch.float64
    _check(ctx.handle, load_library().rpa_pass_begin(ctx.handle, _dev(psi_v, c128), nv, _dev(psi_c, c128), nc, _dev(e_v, f64), _dev(e_c, f64),
                                                     int(nvb), int(n_eig), _dev(omega, f64), n_w, int(bool(keep_m)), int(bool(timing))))
    ctx._pass = dict(refs=(psi_v, psi_c, e_v, e_c, omega), n_eig=int(n_eig), n_w=n_w)


def rpa_pass1_chi0(ctx):
    """{a1, a2} over all valence blocks; returns the partial chi~0(0) [n_g][n_g] as a view into the workspace."""
    import torch
    p = C.c_void_p()
    _check(ctx.handle, load_library().rpa_pass1_chi0(ctx.handle, C.byref(p)))
    return _ws_view(ctx, p.value, torch.complex128, ctx.n_g, ctx.n_g)


def rpa_pass_basis(ctx, tol=0.0, compute=True):
    """a3 on the (reduced) chi~0(0) when `compute`; returns (C [n_eig][n_g], lambda [n_eig]) as views into the workspace."""
    import torch
    pc, pl = C.c_void_p(), C.c_void_p()
    _check(ctx.handle, load_library().rpa_pass_basis(ctx.handle, float(tol), int(bool(compute)), C.byref(pc), C.byref(pl)))
    n_eig = ctx._pass["n_eig"]
    return _ws_view(ctx, pc.value, torch.complex128, n_eig, ctx.n_g), _ws_view(ctx, pl.value, torch.float64, n_eig)


def rpa_pass2_chis(ctx):
    """{a1 unless M was kept, a4} over all valence blocks; returns the partial chi_s [n_w][n_eig][n_eig] (workspace view)."""
    import torch
    p = C.c_void_p()
    _check(ctx.handle, load_library().rpa_pass2_chis(ctx.handle, C.byref(p)))
    n_eig, n_w = ctx._pass["n_eig"], ctx._pass["n_w"]
    return _ws_view(ctx, p.value, torch.complex128, n_w, n_eig, n_eig)


def rpa_pass_energy(ctx, weight):
    """a5 on the (reduced) chi_s; same dict as rpa_energy_device."""
    import torch
    n_eig, n_w = ctx._pass["n_eig"], ctx._pass["n_w"]
    _shape("weight", weight, n_w)
    e = C.c_double(0.0)
    lam = (C.c_double * n_eig)()
    per = (C.c_double * n_w)()
    ms = (C.c_double * 5)()
    _check(ctx.handle, load_library().rpa_pass_energy(ctx.handle, _dev(weight, torch.float64), C.byref(e), lam, per, ms))
    return dict(E_c=e.value, lam=np.array(lam[:]), t=np.array(per[:]),
                stage_ms=dict(zip(("mtxel", "chi0_static", "basis", "chi_freq", "energy"), ms[:])))


def rpa_pass_end(ctx):
    _check(ctx.handle, load_library().rpa_pass_end(ctx.handle))
    ctx._pass = None


def rpa_fp64_peak(ctx, kind: int, iters: int = 20) -> float:
    t = C.c_double(0.0)
    _check(ctx.handle, load_library().rpa_fp64_peak(ctx.handle, kind, iters, C.byref(t)))
    return t.value


def rpa_launch_count(ctx) -> int:
    return int(load_library().rpa_launch_count(ctx.handle))


PROFILE_CLASSES = ("mtxel_plane", "mtxel_z", "mtxel_wfn", "chi0", "proj", "chis", "basis", "energy")


def rpa_profile_begin(ctx):
    _check(ctx.handle, load_library().rpa_profile_begin(ctx.handle))


def rpa_profile_end(ctx):
    """{class: (device ms, timed launches)} for the calls since rpa_profile_begin."""
    n = len(PROFILE_CLASSES)
    ms = (C.c_double * n)()
    cnt = (C.c_longlong * n)()
    _check(ctx.handle, load_library().rpa_profile_end(ctx.handle, ms, cnt))
    return {k: (ms[i], int(cnt[i])) for i, k in enumerate(PROFILE_CLASSES)}


def rpa_basis_info(ctx):
    """(n, sweeps, kind) of the last Jacobi eigen-decomposition of the basis stage (kind 0 vector, 1 block)."""
    n, sw, kind = C.c_int(0), C.c_int(0), C.c_int(0)
    _check(ctx.handle, load_library().rpa_basis_info(ctx.handle, C.byref(n), C.byref(sw), C.byref(kind)))
    return n.value, sw.value, kind.value


def rpa_basis_quality(ctx):
    """(residual, orthogonality) the last basis stage measured on its result: max_i ||chi0 c_i - lambda_i c_i|| / |lambda_1|
    and max |C C^H - 1|."""
    r, o = C.c_double(0.0), C.c_double(0.0)
    _check(ctx.handle, load_library().rpa_basis_quality(ctx.handle, C.byref(r), C.byref(o)))
    return r.value, o.value
