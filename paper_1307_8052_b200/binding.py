"""Thin Python binding of librpa_chi0.so (include/rpa_chi0.h): same names, argument marshalling only.

PyTorch is used for device memory (the workspace and the caller's tensors) and for the CUDA stream; every step
of the path runs in the library's kernels.  There is no CPU fallback: if the shared library is missing or no
CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

RPA_OK = 0
RPA_ERR_INVALID_ARG = -1
RPA_ERR_UNSUPPORTED = -2
RPA_ERR_WORKSPACE = -3
RPA_ERR_CUDA = -4
RPA_ERR_NOT_PD = -5

EXPORTS = (
    "rpa_chi0_workspace_bytes", "rpa_chi0_create", "rpa_chi0_ng", "rpa_chi0_gvectors", "rpa_chi0_add_kpoint",
    "rpa_chi0_get", "rpa_ec_q", "rpa_chi0_reset", "rpa_chi0_sync", "rpa_chi0_set_profiling", "rpa_chi0_stage_times",
    "rpa_chi0_launch_count", "rpa_chi0_accumulators", "rpa_chi0_destroy", "rpa_last_error",
    "rpa_pw_to_grid", "rpa_symmetry_remap", "rpa_momentum_pw", "rpa_chi0_add_kpoint_optical",
    "rpa_chi0_set_spin_degeneracy", "rpa_chi0_create_real_axis", "rpa_ec_q_range",
    "rpa_chi0_set_rank_k_mode", "rpa_chi0_rank_k_batches", "rpa_chi0_set_ec_lanes", "rpa_total_energy",
    "rpa_e_omega_noalloc", "rpa_chi0_add_kpoint_begin", "rpa_chi0_add_kpoint_pairs", "rpa_chi0_add_kpoint_end",
)

# rpa_chi0_set_rank_k_mode (include/rpa_chi0.h)
RPA_RANK_K_FP64_3M = 0
RPA_RANK_K_FP64_4M = 1
RPA_RANK_K_I8 = 2
RPA_RANK_K_FLAG_NO_CLUSTER = 0x100
RPA_RANK_K_FLAG_ALL_BATCHES = 0x200
RPA_EC_FLAG_WIDE_TILES = 0x100   # rpa_chi0_set_ec_lanes

STAGE_NAMES = ("pair_product_fft_yz", "fft_x_gather", "paw", "weights", "rank_k", "rank_k_i8_mma")


class RpaError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"librpa_chi0 error {code}: {msg}")
        self.code = code


_lib = None


def library_path() -> str:
    return _build.LIB


def lib():
    """Load librpa_chi0.so (building it first if nvcc is here and the sources are newer); raises if impossible."""
    global _lib
    if _lib is not None:
        return _lib
    try:
        path = _build.build()
    except Exception as exc:  # no nvcc / compile error: never fall back to anything else
        if not os.path.exists(_build.LIB):
            raise ImportError(f"librpa_chi0.so is missing and could not be built: {exc}") from exc
        path = _build.LIB
    L = C.CDLL(path)
    i32, i64, f64, vp, sz = C.c_int32, C.c_int64, C.c_double, C.c_void_p, C.c_size_t
    L.rpa_chi0_workspace_bytes.restype = sz
    L.rpa_chi0_workspace_bytes.argtypes = [vp, vp, vp, f64, i32, i32, i32]
    L.rpa_chi0_create.restype = C.c_int
    L.rpa_chi0_create.argtypes = [C.POINTER(vp), vp, vp, vp, f64, i32, vp, vp, i32, i32, vp, sz, vp]
    L.rpa_chi0_create_real_axis.restype = C.c_int
    L.rpa_chi0_create_real_axis.argtypes = [C.POINTER(vp), vp, vp, vp, f64, i32, vp, f64, i32, i32, vp, sz, vp]
    L.rpa_chi0_ng.restype = C.c_int
    L.rpa_chi0_ng.argtypes = [vp, C.POINTER(i32)]
    L.rpa_chi0_gvectors.restype = C.c_int
    L.rpa_chi0_gvectors.argtypes = [vp, vp, vp]
    L.rpa_chi0_add_kpoint.restype = C.c_int
    L.rpa_chi0_add_kpoint.argtypes = [vp, f64, i32, vp, i32, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp]
    L.rpa_chi0_add_kpoint_begin.restype = C.c_int
    L.rpa_chi0_add_kpoint_begin.argtypes = L.rpa_chi0_add_kpoint.argtypes
    L.rpa_chi0_add_kpoint_pairs.restype = C.c_int
    L.rpa_chi0_add_kpoint_pairs.argtypes = [vp, i32, i32]
    L.rpa_chi0_add_kpoint_end.restype = C.c_int
    L.rpa_chi0_add_kpoint_end.argtypes = [vp]
    L.rpa_chi0_get.restype = C.c_int
    L.rpa_chi0_get.argtypes = [vp, i32, vp]
    L.rpa_ec_q.restype = C.c_int
    L.rpa_ec_q.argtypes = [vp, vp, C.POINTER(f64), vp]
    L.rpa_ec_q_range.restype = C.c_int
    L.rpa_ec_q_range.argtypes = [vp, vp, i32, i32, C.POINTER(f64), vp]
    for name in ("rpa_chi0_reset", "rpa_chi0_sync"):
        getattr(L, name).restype = C.c_int
        getattr(L, name).argtypes = [vp]
    L.rpa_chi0_set_profiling.restype = C.c_int
    L.rpa_chi0_set_profiling.argtypes = [vp, i32]
    L.rpa_chi0_stage_times.restype = C.c_int
    L.rpa_chi0_stage_times.argtypes = [vp, vp, vp]
    L.rpa_chi0_launch_count.restype = C.c_int
    L.rpa_chi0_launch_count.argtypes = [vp, C.POINTER(i64)]
    L.rpa_chi0_accumulators.restype = C.c_int
    L.rpa_chi0_accumulators.argtypes = [vp, C.POINTER(vp), C.POINTER(sz)]
    L.rpa_chi0_destroy.restype = None
    L.rpa_chi0_destroy.argtypes = [vp]
    L.rpa_chi0_set_rank_k_mode.restype = C.c_int
    L.rpa_chi0_set_rank_k_mode.argtypes = [vp, i32, i32]
    L.rpa_chi0_rank_k_batches.restype = C.c_int
    L.rpa_chi0_rank_k_batches.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
    L.rpa_chi0_set_ec_lanes.restype = C.c_int
    L.rpa_chi0_set_ec_lanes.argtypes = [vp, i32]
    L.rpa_total_energy.restype = C.c_int
    L.rpa_total_energy.argtypes = [i32, vp, vp, C.POINTER(f64)]
    L.rpa_e_omega_noalloc.restype = C.c_int
    L.rpa_e_omega_noalloc.argtypes = [vp, i32, vp, vp, vp]
    L.rpa_pw_to_grid.restype = C.c_int
    L.rpa_pw_to_grid.argtypes = [vp, i32, i32, vp, vp, vp]
    L.rpa_symmetry_remap.restype = C.c_int
    L.rpa_symmetry_remap.argtypes = [vp, i32, vp, i32, vp, vp]
    L.rpa_chi0_set_spin_degeneracy.restype = C.c_int
    L.rpa_chi0_set_spin_degeneracy.argtypes = [vp, i32]
    L.rpa_momentum_pw.restype = C.c_int
    L.rpa_momentum_pw.argtypes = [vp, vp, i32, vp, i32, vp, i32, vp, i32, vp, vp, vp, vp, vp]
    L.rpa_chi0_add_kpoint_optical.restype = C.c_int
    L.rpa_chi0_add_kpoint_optical.argtypes = [vp, f64, i32, vp, i32, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp]
    L.rpa_last_error.restype = C.c_char_p
    L.rpa_last_error.argtypes = []
    _lib = L
    return L


def _check(rc: int):
    if rc != RPA_OK:
        raise RpaError(rc, lib().rpa_last_error().decode("utf-8", "replace"))


def rpa_last_error() -> str:
    return lib().rpa_last_error().decode("utf-8", "replace")


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _hp(a) -> C.c_void_p:
    return a.ctypes.data_as(C.c_void_p)


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1307_8052_b200 needs a CUDA device (there is no CPU fallback)")
    return torch


def _dev_ptr(t, name: str, dtype, device) -> C.c_void_p:
    torch = _torch()
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor")
    if t.dtype != dtype:
        raise TypeError(f"{name} must have dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if t.device != device:
        raise ValueError(f"{name} is on {t.device}, the handle on {device}")
    return C.c_void_p(t.data_ptr())


class Handle:
    """Owns the opaque rpa_chi0_t* and the torch-allocated workspace it lives in."""

    def __init__(self, ptr, workspace, device, stream, grid, n_omega):
        self.ptr, self.workspace, self.device, self.stream = ptr, workspace, device, stream
        self.grid, self.n_omega = tuple(int(x) for x in grid), int(n_omega)
        self._ng = None

    @property
    def ng(self) -> int:
        if self._ng is None:
            self._ng = rpa_chi0_ng(self)
        return self._ng

    def close(self):
        if self.ptr:
            lib().rpa_chi0_destroy(self.ptr)
            self.ptr = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def rpa_chi0_workspace_bytes(grid, cell, q_red, ecut_ha, n_omega, max_batch_pairs=0, max_proj_total=0) -> int:
    g, c, q = _np(grid, np.int32), _np(cell, np.float64).reshape(9), _np(q_red, np.float64)
    n = int(lib().rpa_chi0_workspace_bytes(_hp(g), _hp(c), _hp(q), float(ecut_ha), int(n_omega), int(max_batch_pairs),
                                           int(max_proj_total)))
    if n == 0:
        raise RpaError(RPA_ERR_INVALID_ARG, rpa_last_error())
    return n


def rpa_chi0_create(grid, cell, q_red, ecut_ha, omega_ha, omega_wt=None, max_batch_pairs=0, max_proj_total=0,
                    device="cuda:0", stream=None, eta_ha=None) -> Handle:
    """eta_ha given: rpa_chi0_create_real_axis (omega_ha real frequencies, chi0 at omega + i eta, no omega_wt)."""
    torch = _torch()
    device = torch.device(device)
    if device.index is None:
        device = torch.device("cuda", torch.cuda.current_device())
    g, c, q = _np(grid, np.int32), _np(cell, np.float64).reshape(9), _np(q_red, np.float64)
    om = _np(omega_ha, np.float64)
    wt = None if omega_wt is None else _np(omega_wt, np.float64)
    n_slots = om.size if eta_ha is None else 2 * om.size
    nbytes = rpa_chi0_workspace_bytes(g, c, q, ecut_ha, n_slots, max_batch_pairs, max_proj_total)
    with torch.cuda.device(device):
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
        off = (-ws.data_ptr()) % 256
        if stream is None:
            stream = torch.cuda.current_stream(device)
        out = C.c_void_p()
        if eta_ha is None:
            rc = lib().rpa_chi0_create(C.byref(out), _hp(g), _hp(c), _hp(q), float(ecut_ha), int(om.size), _hp(om),
                                       None if wt is None else _hp(wt), int(max_batch_pairs), int(max_proj_total),
                                       C.c_void_p(ws.data_ptr() + off), C.c_size_t(nbytes), C.c_void_p(stream.cuda_stream))
        else:
            rc = lib().rpa_chi0_create_real_axis(C.byref(out), _hp(g), _hp(c), _hp(q), float(ecut_ha), int(om.size),
                                                 _hp(om), float(eta_ha), int(max_batch_pairs), int(max_proj_total),
                                                 C.c_void_p(ws.data_ptr() + off), C.c_size_t(nbytes),
                                                 C.c_void_p(stream.cuda_stream))
    _check(rc)
    return Handle(out, ws, device, stream, g, om.size)


def rpa_chi0_create_real_axis(grid, cell, q_red, ecut_ha, omega_ha, eta_ha, max_batch_pairs=0, max_proj_total=0,
                              device="cuda:0", stream=None) -> Handle:
    """chi0 at the real frequencies omega_ha + i eta_ha (NEXT-4); rpa_chi0_get then returns a non-Hermitian matrix."""
    return rpa_chi0_create(grid, cell, q_red, ecut_ha, omega_ha, None, max_batch_pairs, max_proj_total, device, stream,
                           eta_ha=float(eta_ha))


def rpa_chi0_ng(h: Handle) -> int:
    n = C.c_int32()
    _check(lib().rpa_chi0_ng(h.ptr, C.byref(n)))
    return int(n.value)


def rpa_chi0_gvectors(h: Handle):
    ng = h.ng
    g = np.zeros((ng, 3), dtype=np.int32)
    K2 = np.zeros(ng, dtype=np.float64)
    _check(lib().rpa_chi0_gvectors(h.ptr, _hp(g), _hp(K2)))
    return g, K2


def rpa_chi0_add_kpoint(h: Handle, kweight, psi_occ, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc,
                        n_proj: Optional[Sequence[int]] = None, P_occ=None, P_unocc=None, Q=None, R_cart=None,
                        qdir_cart=None, grad=None, _begin=False):
    """psi_*, P_*, Q: CUDA complex128 tensors (layouts of include/rpa_chi0.h); eps_*, f_*, n_proj, R_cart: host.
    With qdir_cart and grad (CUDA [3][n_occ][n_unocc]) this is rpa_chi0_add_kpoint_optical (q = 0 handles)."""
    torch = _torch()
    c128 = torch.complex128
    N = int(np.prod(h.grid))
    n_occ = int(psi_occ.shape[0]) if psi_occ.numel() else 0
    n_unocc = int(psi_unocc.shape[0]) if psi_unocc.numel() else 0
    if n_occ and psi_occ.numel() != n_occ * N:
        raise ValueError("psi_occ must be [n_occ][N1][N2][N3]")
    if n_unocc and psi_unocc.numel() != n_unocc * N:
        raise ValueError("psi_unocc must be [n_unocc][N1][N2][N3]")
    eo, eu = _np(eps_occ, np.float64), _np(eps_unocc, np.float64)
    fo, fu = _np(f_occ, np.float64), _np(f_unocc, np.float64)
    if eo.size != n_occ or fo.size != n_occ or eu.size != n_unocc or fu.size != n_unocc:
        raise ValueError("eps/f lengths must match the band counts")
    n_atoms = 0 if n_proj is None else len(n_proj)
    if n_atoms:
        npj = _np(n_proj, np.int32)
        ptot = int(npj.sum())
        R = _np(R_cart, np.float64).reshape(-1)
        if R.size != 3 * n_atoms:
            raise ValueError("R_cart must be [n_atoms][3]")
        if P_occ.numel() != n_occ * ptot or P_unocc.numel() != n_unocc * ptot:
            raise ValueError("P_occ / P_unocc must be [bands][sum n_proj]")
        if Q.numel() != int((npj.astype(np.int64) ** 2).sum()) * h.ng:
            raise ValueError("Q must hold sum_a n_a^2 * ng elements")
        args = (int(n_atoms), _hp(npj), _dev_ptr(P_occ, "P_occ", c128, h.device) if n_occ else None,
                _dev_ptr(P_unocc, "P_unocc", c128, h.device) if n_unocc else None, _dev_ptr(Q, "Q", c128, h.device), _hp(R))
    else:
        args = (0, None, None, None, None, None)
    common = (h.ptr, float(kweight), n_occ, _dev_ptr(psi_occ, "psi_occ", c128, h.device) if n_occ else None, n_unocc,
              _dev_ptr(psi_unocc, "psi_unocc", c128, h.device) if n_unocc else None, _hp(eo), _hp(eu), _hp(fo), _hp(fu), *args)
    if _begin:
        rc = lib().rpa_chi0_add_kpoint_begin(*common)
    elif grad is None and qdir_cart is None:
        rc = lib().rpa_chi0_add_kpoint(*common)
    else:
        if grad is None or qdir_cart is None or grad.numel() != 3 * n_occ * n_unocc:
            raise ValueError("optical limit: qdir_cart and grad [3][n_occ][n_unocc] are both required")
        qd = _np(qdir_cart, np.float64).reshape(3)
        rc = lib().rpa_chi0_add_kpoint_optical(*common, _hp(qd), _dev_ptr(grad, "grad", c128, h.device))
    _check(rc)


def rpa_chi0_add_kpoint_begin(h: Handle, kweight, psi_occ, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc, n_proj=None,
                              P_occ=None, P_unocc=None, Q=None, R_cart=None):
    """Open a k-point whose unoccupied orbitals (rows of psi_unocc) are still being produced on the handle's stream:
    followed by rpa_chi0_add_kpoint_pairs for consecutive band slices and rpa_chi0_add_kpoint_end.  RpaError with code
    RPA_ERR_UNSUPPORTED when the transitions do not fit one batch (then use rpa_chi0_add_kpoint)."""
    rpa_chi0_add_kpoint(h, kweight, psi_occ, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc, n_proj, P_occ, P_unocc, Q, R_cart,
                        _begin=True)


def rpa_chi0_add_kpoint_pairs(h: Handle, m_begin: int, m_end: int):
    _check(lib().rpa_chi0_add_kpoint_pairs(h.ptr, int(m_begin), int(m_end)))


def rpa_chi0_add_kpoint_end(h: Handle):
    _check(lib().rpa_chi0_add_kpoint_end(h.ptr))


def rpa_chi0_get(h: Handle, i_omega: int, out=None):
    torch = _torch()
    ng = h.ng
    if out is None:
        out = torch.empty((ng, ng), dtype=torch.complex128, device=h.device)
    elif tuple(out.shape) != (ng, ng):
        raise ValueError("out must be [ng][ng]")
    _check(lib().rpa_chi0_get(h.ptr, int(i_omega), _dev_ptr(out, "out", torch.complex128, h.device)))
    return out


def rpa_ec_q(h: Handle, v_G):
    v = _np(v_G, np.float64)
    if v.size != h.ng:
        raise ValueError("v_G must have ng entries")
    ec = C.c_double(0.0)
    e = np.zeros(h.n_omega, dtype=np.float64)
    _check(lib().rpa_ec_q(h.ptr, _hp(v), C.byref(ec), _hp(e)))
    return float(ec.value), e


def rpa_ec_q_range(h: Handle, v_G, iw_begin: int, iw_end: int):
    """(partial E_c(q) of the frequencies [iw_begin, iw_end), their e(omega)); the partial values of disjoint ranges
    covering all frequencies add up to E_c(q)."""
    v = _np(v_G, np.float64)
    if v.size != h.ng:
        raise ValueError("v_G must have ng entries")
    ec = C.c_double(0.0)
    e = np.zeros(max(0, int(iw_end) - int(iw_begin)), dtype=np.float64)
    _check(lib().rpa_ec_q_range(h.ptr, _hp(v), int(iw_begin), int(iw_end), C.byref(ec), _hp(e) if e.size else None))
    return float(ec.value), e


def rpa_chi0_reset(h: Handle):
    _check(lib().rpa_chi0_reset(h.ptr))


def rpa_chi0_set_spin_degeneracy(h: Handle, s: int):
    _check(lib().rpa_chi0_set_spin_degeneracy(h.ptr, int(s)))


def rpa_total_energy(ec_q, q_weights) -> float:
    """E_c = sum_q w_q E_c(q) (Eq. 1): the outer q loop's final sum over the IBZ weights, by the library."""
    e, w = _np(ec_q, np.float64).reshape(-1), _np(q_weights, np.float64).reshape(-1)
    if e.shape != w.shape:
        raise ValueError("one weight per q-point")
    out = C.c_double(0.0)
    _check(lib().rpa_total_energy(int(e.size), _hp(e), _hp(w), C.byref(out)))
    return float(out.value)


RPA_NOALLOC_MAX_NG = 512


def rpa_e_omega_noalloc(chi0, v_G, e, stream=None):
    """e[0] = ln det(1 - v^1/2 chi0 v^1/2) + Tr(v^1/2 chi0 v^1/2) (Eq. 2's integrand) for one DEVICE matrix chi0 [ng][ng]
    complex128, v_G a DEVICE double [ng], e a DEVICE double [1]; asynchronous on `stream` (a torch.cuda.Stream; None =
    torch's current stream).  No device allocation: the scratch is a fixed array of the library (ng <= 512)."""
    torch = _torch()
    if not isinstance(chi0, torch.Tensor) or chi0.dim() != 2 or chi0.shape[0] != chi0.shape[1]:
        raise ValueError("chi0 must be a square CUDA tensor")
    ng, dev = int(chi0.shape[0]), chi0.device
    if tuple(v_G.shape) != (ng,) or e.numel() != 1:
        raise ValueError("v_G must be [ng], e one double")
    st = torch.cuda.current_stream(dev) if stream is None else stream
    with torch.cuda.device(dev):
        _check(lib().rpa_e_omega_noalloc(_dev_ptr(chi0, "chi0", torch.complex128, dev), ng,
                                         _dev_ptr(v_G, "v_G", torch.float64, dev), _dev_ptr(e, "e", torch.float64, dev),
                                         C.c_void_p(st.cuda_stream)))


def rpa_chi0_set_rank_k_mode(h: Handle, mode: int, digits: int = 0):
    """mode: RPA_RANK_K_FP64_3M (default of the library) / RPA_RANK_K_FP64_4M / RPA_RANK_K_I8 [| RPA_RANK_K_FLAG_*]."""
    _check(lib().rpa_chi0_set_rank_k_mode(h.ptr, int(mode), int(digits)))


def rpa_chi0_rank_k_batches(h: Handle):
    """(batches run on the FP64 tensor kernels, batches run on the int8-sliced kernel) since create."""
    a, b = C.c_int64(0), C.c_int64(0)
    _check(lib().rpa_chi0_rank_k_batches(h.ptr, C.byref(a), C.byref(b)))
    return int(a.value), int(b.value)


def rpa_chi0_set_ec_lanes(h: Handle, n_lanes: int):
    _check(lib().rpa_chi0_set_ec_lanes(h.ptr, int(n_lanes)))


def rpa_chi0_sync(h: Handle):
    _check(lib().rpa_chi0_sync(h.ptr))


def rpa_chi0_set_profiling(h: Handle, on: bool):
    _check(lib().rpa_chi0_set_profiling(h.ptr, 1 if on else 0))


def rpa_chi0_stage_times(h: Handle):
    ms = np.zeros(6, dtype=np.float64)
    n = np.zeros(6, dtype=np.int64)
    _check(lib().rpa_chi0_stage_times(h.ptr, _hp(ms), _hp(n)))
    return ms, n


def rpa_chi0_launch_count(h: Handle) -> int:
    n = C.c_int64(0)
    _check(lib().rpa_chi0_launch_count(h.ptr, C.byref(n)))
    return int(n.value)


def rpa_chi0_accumulators(h: Handle):
    """The accumulators as a flat complex128 CUDA tensor aliasing the workspace (for an in-place all-reduce)."""
    torch = _torch()
    p, n = C.c_void_p(), C.c_size_t()
    _check(lib().rpa_chi0_accumulators(h.ptr, C.byref(p), C.byref(n)))
    off = int(p.value) - h.workspace.data_ptr()
    return h.workspace[off:off + int(n.value)].view(torch.complex128)


def rpa_pw_to_grid(h: Handle, g_pw, C_pw, out=None):
    """Eq. 10: C_pw CUDA complex128 [n_bands][n_pw], g_pw host int [n_pw][3] -> psi [n_bands][N1][N2][N3] (CUDA)."""
    torch = _torch()
    g = _np(g_pw, np.int32).reshape(-1, 3)
    n_pw = g.shape[0]
    if C_pw.dim() != 2 or int(C_pw.shape[1]) != n_pw:
        raise ValueError("C_pw must be [n_bands][n_pw]")
    n_bands = int(C_pw.shape[0])
    if out is None:
        out = torch.empty((n_bands,) + h.grid, dtype=torch.complex128, device=h.device)
    elif out.numel() != n_bands * int(np.prod(h.grid)):
        raise ValueError("out must be [n_bands][N1][N2][N3]")
    _check(lib().rpa_pw_to_grid(h.ptr, n_bands, n_pw, _hp(g), _dev_ptr(C_pw, "C_pw", torch.complex128, h.device) if n_bands else None,
                                _dev_ptr(out, "out", torch.complex128, h.device) if n_bands else None))
    return out


def rpa_symmetry_remap(h: Handle, psi, M, time_reversal=False, out=None):
    """Eq. 11: psi_out(r) = psi(M r) in reduced coordinates (M = T^-1, integer 3x3), conjugated under time reversal."""
    torch = _torch()
    Mi = _np(M, np.int32).reshape(9)
    N = int(np.prod(h.grid))
    n_bands = psi.numel() // N
    if out is None:
        out = torch.empty_like(psi)
    _check(lib().rpa_symmetry_remap(h.ptr, n_bands, _hp(Mi), 1 if time_reversal else 0,
                                    _dev_ptr(psi, "psi", torch.complex128, h.device), _dev_ptr(out, "out", torch.complex128, h.device)))
    return out


def rpa_chi0_add_kpoint_optical(h: Handle, kweight, psi_occ, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc, qdir_cart, grad,
                                n_proj=None, P_occ=None, P_unocc=None, Q=None, R_cart=None):
    rpa_chi0_add_kpoint(h, kweight, psi_occ, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc, n_proj, P_occ, P_unocc, Q, R_cart,
                        qdir_cart, grad)


def rpa_momentum_pw(h: Handle, k_cart, g_pw, C_occ, C_unocc, n_proj=None, P_occ=None, P_unocc=None, Qgrad=None):
    """Eq. 15 / 19: grad[3][n_occ][n_unocc] (CUDA) from plane-wave coefficients C_* (CUDA [bands][n_pw]) + PAW term."""
    torch = _torch()
    c128 = torch.complex128
    g = _np(g_pw, np.int32).reshape(-1, 3)
    k = _np(k_cart, np.float64).reshape(3)
    n_pw = g.shape[0]
    n_occ, n_unocc = int(C_occ.shape[0]), int(C_unocc.shape[0])
    if int(C_occ.shape[1]) != n_pw or int(C_unocc.shape[1]) != n_pw:
        raise ValueError("C_occ / C_unocc must be [bands][n_pw]")
    out = torch.empty((3, n_occ, n_unocc), dtype=c128, device=h.device)
    if n_proj is not None and len(n_proj):
        npj = _np(n_proj, np.int32)
        paw = (len(npj), _hp(npj), _dev_ptr(P_occ, "P_occ", c128, h.device), _dev_ptr(P_unocc, "P_unocc", c128, h.device),
               _dev_ptr(Qgrad, "Qgrad", c128, h.device))
    else:
        paw = (0, None, None, None, None)
    _check(lib().rpa_momentum_pw(h.ptr, _hp(k), n_pw, _hp(g), n_occ, _dev_ptr(C_occ, "C_occ", c128, h.device), n_unocc,
                                 _dev_ptr(C_unocc, "C_unocc", c128, h.device), *paw, _dev_ptr(out, "grad", c128, h.device)))
    return out


def rpa_chi0_destroy(h: Handle):
    h.close()


# ---- host-buffer convenience on top of the calls above (the end-to-end path bench.py times) ------------------

def add_kpoint_host(h: Handle, kd, n_proj=None, Q_dev=None, R_cart=None, pinned=None, kweight=None, chunk_bands=64):
    """Copy one k-point's host arrays (workload.KPointData) to the device and add it; returns the bytes copied
    host->device.  `pinned` may hold pre-pinned host tensors keyed like the KPointData fields.

    The unoccupied orbitals (the bulk of the bytes) are uploaded in slices of `chunk_bands` bands on a side stream
    into two alternating device buffers, and every slice is added with its own rpa_chi0_add_kpoint call (the
    accumulation is additive over any split of the bands), so the copy of slice i+1 overlaps the
    kernels of slice i.  Only marshalling happens here: all arithmetic is in the library."""
    torch = _torch()
    dev = h.device

    def host(name):
        return pinned[name] if pinned is not None else torch.from_numpy(getattr(kd, name))

    kw = kd.kweight if kweight is None else kweight
    have_paw = n_proj is not None and len(n_proj) > 0
    main = h.stream
    with torch.cuda.device(dev), torch.cuda.stream(main):
        psi_o = host("psi_occ").to(dev, non_blocking=True)
        nbytes = psi_o.numel() * 16
        P_o = P_u = None
        if have_paw:
            P_o, P_u = host("P_occ").to(dev, non_blocking=True), host("P_unocc").to(dev, non_blocking=True)
            nbytes += P_o.numel() * 16 + P_u.numel() * 16
        src = host("psi_unocc")
        n_un = int(src.shape[0])
        nbytes += src.numel() * 16
        if n_un <= chunk_bands or not src.is_pinned():
            psi_u = src.to(dev, non_blocking=True)
            rpa_chi0_add_kpoint(h, kw, psi_o, psi_u, kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc, n_proj, P_o, P_u,
                                Q_dev, R_cart)
            return nbytes
        side = getattr(h, "_copy_stream", None)
        if side is None:
            side = h._copy_stream = torch.cuda.Stream(device=dev)
        bufs = [torch.empty((chunk_bands,) + tuple(src.shape[1:]), dtype=src.dtype, device=dev) for _ in range(2)]
        free = [None, None]   # event: the kernels that read this buffer have been enqueued and finished
        side.wait_stream(main)   # the buffers were allocated on the main stream
        for i, m0 in enumerate(range(0, n_un, chunk_bands)):
            m1 = min(m0 + chunk_bands, n_un)
            b = i & 1
            with torch.cuda.stream(side):
                if free[b] is not None:
                    side.wait_event(free[b])
                bufs[b][:m1 - m0].copy_(src[m0:m1], non_blocking=True)
                ready = torch.cuda.Event()
                ready.record(side)
            main.wait_event(ready)
            rpa_chi0_add_kpoint(h, kw, psi_o, bufs[b][:m1 - m0], kd.eps_occ, kd.eps_unocc[m0:m1], kd.f_occ,
                                kd.f_unocc[m0:m1], n_proj, P_o, None if P_u is None else P_u[m0:m1].contiguous(),
                                Q_dev, R_cart)
            free[b] = torch.cuda.Event()
            free[b].record(main)
        side.wait_stream(main)   # the buffers may be released once the main stream has passed this point
    return nbytes


def add_kpoint_host_pw(h: Handle, kweight, g_pw, C_occ, C_unocc, eps_occ, eps_unocc, f_occ, f_unocc, n_proj=None,
                       P_occ=None, P_unocc=None, Q_dev=None, R_cart=None, n_slices=8, n_calls=1, streamed=True):
    """The paper's own pipeline (Table 1 steps 3 and 5-11): the host holds the orbitals as plane-wave coefficients
    C_*[bands][n_pw] (host tensors, ideally pinned; g_pw[n_pw][3] their integer wave vectors) -- about 1/20 of the
    bytes of the grid orbitals -- the device expands them with rpa_pw_to_grid (Eq. 10) into buffers kept on the
    handle and adds the k-point.  Returns the bytes copied host->device.  Marshalling only.

    The coefficients go up on a side stream, the unoccupied ones in `n_slices` slices; rpa_pw_to_grid of a slice is
    enqueued on the handle's stream behind the event of its copy, so the expansion of slice i runs under the copy of
    slice i + 1 (rpa_pw_to_grid keeps the index table of g_pw on the device between calls and does not block).  When the
    transitions fit one batch the k-point is added with rpa_chi0_add_kpoint_begin / _pairs / _end: the pair densities of a
    slice are enqueued right behind its expansion, so the remaining uploads hide under them and only the first slice's
    copy is exposed; the result is that of one rpa_chi0_add_kpoint call, bit for bit.  Otherwise (or with n_calls > 1)
    the unoccupied bands are added in `n_calls` rpa_chi0_add_kpoint calls after their slices have arrived (the accumulation
    is additive over any split of the bands)."""
    torch = _torch()
    dev = h.device
    have_paw = n_proj is not None and len(n_proj) > 0
    main = h.stream
    with torch.cuda.device(dev), torch.cuda.stream(main):
        t = lambda a: a if isinstance(a, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(a))
        C_oh, C_uh = t(C_occ), t(C_unocc)
        n_o, n_u, n_pw = int(C_oh.shape[0]), int(C_uh.shape[0]), int(C_oh.shape[1])
        nbytes = (C_oh.numel() + C_uh.numel()) * 16
        P_oh = P_uh = None
        if have_paw:
            P_oh, P_uh = t(P_occ), t(P_unocc)
            nbytes += (P_oh.numel() + P_uh.numel()) * 16
        key = (n_o, n_u, n_pw, 0 if P_oh is None else int(P_oh.shape[1]))
        bufs = getattr(h, "_pw_bufs", None)
        if bufs is None or bufs["key"] != key:
            c128 = dict(dtype=torch.complex128, device=dev)
            bufs = h._pw_bufs = {"key": key, "psi_o": torch.empty((n_o,) + h.grid, **c128), "psi_u": torch.empty((n_u,) + h.grid, **c128),
                                 "C_o": torch.empty((n_o, n_pw), **c128), "C_u": torch.empty((n_u, n_pw), **c128),
                                 "P_o": None if P_oh is None else torch.empty(tuple(P_oh.shape), **c128),
                                 "P_u": None if P_uh is None else torch.empty(tuple(P_uh.shape), **c128)}
        side = getattr(h, "_copy_stream", None)
        if side is None:
            side = h._copy_stream = torch.cuda.Stream(device=dev)
        side.wait_stream(main)   # the kernels of the previous call that read these buffers are enqueued on the main stream

        def upload(dst, src):
            with torch.cuda.stream(side):
                dst.copy_(src, non_blocking=True)
                ev = torch.cuda.Event()
                ev.record(side)
            return ev

        ev = upload(bufs["C_o"], C_oh)
        main.wait_event(ev)
        rpa_pw_to_grid(h, g_pw, bufs["C_o"], bufs["psi_o"])
        if have_paw:
            upload(bufs["P_o"], P_oh)
            main.wait_event(upload(bufs["P_u"], P_uh))
        eps_u, f_u = _np(eps_unocc, np.float64), _np(f_unocc, np.float64)
        n_calls = max(1, min(int(n_calls), n_u))
        want_streamed, streamed = bool(streamed), False
        if want_streamed and n_calls == 1 and n_u > 1:
            # one k-point, its pair densities slice by slice as the orbitals arrive (rpa_chi0_add_kpoint_begin / _pairs / _end)
            try:
                rpa_chi0_add_kpoint_begin(h, kweight, bufs["psi_o"], bufs["psi_u"], eps_occ, eps_u, f_occ, f_u, n_proj, bufs["P_o"],
                                          bufs["P_u"], Q_dev, R_cart)
                streamed = True
            except RpaError as e:
                if e.code != RPA_ERR_UNSUPPORTED:
                    raise
        per_call = max(1, -(-n_u // n_calls))
        step = max(1, -(-per_call // max(1, int(n_slices) // n_calls)))
        for c0 in range(0, n_u, per_call):
            c1 = min(c0 + per_call, n_u)
            for m0 in range(c0, c1, step):
                m1 = min(m0 + step, c1)
                ev = upload(bufs["C_u"][m0:m1], C_uh[m0:m1])
                main.wait_event(ev)
                rpa_pw_to_grid(h, g_pw, bufs["C_u"][m0:m1], bufs["psi_u"][m0:m1])
                if streamed:
                    rpa_chi0_add_kpoint_pairs(h, m0, m1)
            if streamed:
                rpa_chi0_add_kpoint_end(h)
            else:
                rpa_chi0_add_kpoint(h, kweight, bufs["psi_o"], bufs["psi_u"][c0:c1], eps_occ, eps_u[c0:c1], f_occ, f_u[c0:c1], n_proj,
                                    bufs["P_o"], None if bufs["P_u"] is None else bufs["P_u"][c0:c1], Q_dev, R_cart)
    return nbytes
