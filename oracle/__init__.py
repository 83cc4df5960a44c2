"""CPU ORACLE (test infrastructure only) -- ctypes front end of oracle/rpa_oracle.c.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` / ``--impl reference`` legs may import
this package.  It imports nothing from ``paper_1307_8052_b200`` and shares no code with the CUDA path.
Every routine here is pinned by tests/test_oracle_pins.py; none is "parity unpinned".

``Chi0Oracle`` strings the C routines together in the paper's order (Table 1 steps 5, 6, 8, 9, 11, 13;
P:L149-162) with the same call shape as the library boundary, so a test can feed both the same arrays.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        i32, f64, vp = C.c_int32, C.c_double, C.c_void_p
        L.orc_num_threads.restype = i32
        L.orc_volume.restype = f64
        L.orc_volume.argtypes = [vp]
        L.orc_sphere.restype = i32
        L.orc_sphere.argtypes = [vp, vp, vp, f64, i32, vp, vp]
        L.orc_K2.restype = None
        L.orc_K2.argtypes = [vp, vp, i32, vp, vp]
        for name in ("orc_pair_density_naive", "orc_pair_density_separable"):
            f = getattr(L, name)
            f.restype = None
            f.argtypes = [vp, vp, i32, vp, i32, vp, vp]
        L.orc_paw_add.restype = None
        L.orc_paw_add.argtypes = [vp, vp, i32, vp, i32, vp, vp, i32, vp, vp, vp, vp]
        L.orc_weights.restype = None
        L.orc_weights.argtypes = [f64, f64, i32, vp, vp, i32, vp, vp]
        L.orc_accumulate.restype = None
        L.orc_accumulate.argtypes = [i32, i32, vp, i32, vp, f64, vp]
        L.orc_weights_z.restype = None
        L.orc_weights_z.argtypes = [f64, f64, i32, vp, vp, i32, vp, vp]
        L.orc_accumulate_z.restype = None
        L.orc_accumulate_z.argtypes = [i32, i32, vp, i32, vp, f64, vp]
        L.orc_chi0_from_S.restype = None
        L.orc_chi0_from_S.argtypes = [C.c_int64, f64, vp, vp]
        L.orc_ec_q.restype = i32
        L.orc_ec_q.argtypes = [i32, i32, vp, vp, vp, vp, vp]
        L.orc_chi0_from_S_spin.restype = None
        L.orc_chi0_from_S_spin.argtypes = [C.c_int64, f64, f64, vp, vp]
        L.orc_pw_to_grid.restype = None
        L.orc_pw_to_grid.argtypes = [vp, i32, i32, vp, vp, C.c_int64, vp, vp]
        L.orc_symmetry_remap.restype = i32
        L.orc_symmetry_remap.argtypes = [vp, vp, i32, i32, vp, vp]
        L.orc_momentum_pw.restype = None
        L.orc_momentum_pw.argtypes = [vp, vp, i32, vp, i32, vp, i32, vp, i32, vp, vp, vp, vp, vp]
        L.orc_optical_head.restype = None
        L.orc_optical_head.argtypes = [i32, i32, vp, vp, vp, vp, vp]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def volume(cell) -> float:
    return float(lib().orc_volume(_p(_f64(cell).reshape(9))))


def sphere(grid, cell, q_red, ecut_ha):
    """(g[ng,3] int32, K2[ng]) in ascending flat-FFT-index order."""
    grid, cell, q = _i32(grid), _f64(cell).reshape(9), _f64(q_red)
    ng = lib().orc_sphere(_p(grid), _p(cell), _p(q), float(ecut_ha), 0, None, None)
    g = np.zeros((ng, 3), dtype=np.int32)
    K2 = np.zeros(ng, dtype=np.float64)
    lib().orc_sphere(_p(grid), _p(cell), _p(q), float(ecut_ha), ng, _p(g), _p(K2))
    return g, K2


def K2_of(cell, q_red, g):
    g = _i32(g).reshape(-1, 3)
    out = np.zeros(g.shape[0], dtype=np.float64)
    lib().orc_K2(_p(_f64(cell).reshape(9)), _p(_f64(q_red)), g.shape[0], _p(g), _p(out))
    return out


def pair_density(grid, u_n, u_m, g, mode="separable"):
    """ntilde[m][g] for one u_n against a stack u_m[n_m][N1][N2][N3]."""
    grid = _i32(grid)
    u_n, u_m, g = _c128(u_n), _c128(u_m), _i32(g).reshape(-1, 3)
    N = int(np.prod(grid))
    n_m = u_m.size // N
    out = np.zeros((n_m, g.shape[0]), dtype=np.complex128)
    fn = {"separable": lib().orc_pair_density_separable, "naive": lib().orc_pair_density_naive}[mode]
    fn(_p(grid), _p(u_n), n_m, _p(u_m), g.shape[0], _p(g), _p(out))
    return out


def paw_add(cell, q_red, g, n_proj, P_n, P_m, Q, R_cart, n):
    """In-place n[m][g] += PAW term; returns n."""
    g = _i32(g).reshape(-1, 3)
    n_proj = _i32(n_proj)
    P_n, P_m, Q, R = _c128(P_n), _c128(P_m), _c128(Q), _f64(R_cart)
    assert n.dtype == np.complex128 and n.flags.c_contiguous
    n_m = n.shape[0]
    lib().orc_paw_add(_p(_f64(cell).reshape(9)), _p(_f64(q_red)), g.shape[0], _p(g), n_proj.size, _p(n_proj), _p(P_n),
                      n_m, _p(P_m), _p(Q), _p(R), _p(n))
    return n


def weights(eps_n, f_n, eps_m, f_m, omega):
    eps_m, f_m, omega = _f64(eps_m), _f64(f_m), _f64(omega)
    w = np.zeros((omega.size, eps_m.size), dtype=np.float64)
    lib().orc_weights(float(eps_n), float(f_n), eps_m.size, _p(eps_m), _p(f_m), omega.size, _p(omega), _p(w))
    return w


def accumulate(S, n, w, kweight):
    """S[nw][ng][ng] += kweight * sum_p w[iw][p] n[p][g] conj(n[p][g'])."""
    n, w = _c128(n), _f64(w)
    assert S.dtype == np.complex128 and S.flags.c_contiguous
    lib().orc_accumulate(n.shape[1], n.shape[0], _p(n), w.shape[0], _p(w), float(kweight), _p(S))
    return S


def weights_z(eps_n, f_n, eps_m, f_m, z):
    """Complex weights of Eq. 3 at the complex frequencies z (NEXT-4 real axis: z = omega + i eta): [iz][m]."""
    eps_m, f_m, z = _f64(eps_m), _f64(f_m), _c128(z)
    w = np.zeros((z.size, eps_m.size), dtype=np.complex128)
    lib().orc_weights_z(float(eps_n), float(f_n), eps_m.size, _p(eps_m), _p(f_m), z.size, _p(z), _p(w))
    return w


def accumulate_z(S, n, w, kweight):
    """S[nz][ng][ng] += kweight * sum_p w[iz][p] n[p][g] conj(n[p][g']) with complex w."""
    n, w = _c128(n), _c128(w)
    assert S.dtype == np.complex128 and S.flags.c_contiguous
    lib().orc_accumulate_z(n.shape[1], n.shape[0], _p(n), w.shape[0], _p(w), float(kweight), _p(S))
    return S


def chi0_from_S(S, vol, spin_deg=None):
    """chi0 = (2/Omega) S (spin-paired, reading A3), or (spin_deg/Omega) S for explicit spin channels (NEXT-4)."""
    S = _c128(S)
    out = np.empty_like(S)
    if spin_deg is None:
        lib().orc_chi0_from_S(S.size, float(vol), _p(S), _p(out))
    else:
        lib().orc_chi0_from_S_spin(S.size, float(vol), float(spin_deg), _p(S), _p(out))
    return out


def ec_q(chi0, v, omega_wt):
    """(E_c(q), e_omega[nw]); raises if I - D chi0 D is not positive definite."""
    chi0, v, wt = _c128(chi0), _f64(v), _f64(omega_wt)
    nw, ng = chi0.shape[0], chi0.shape[1]
    ec = C.c_double(0.0)
    e = np.zeros(nw, dtype=np.float64)
    st = lib().orc_ec_q(ng, nw, _p(chi0), _p(v), _p(wt), C.byref(ec), _p(e))
    if st != 0:
        raise FloatingPointError(f"I - v^1/2 chi0 v^1/2 not positive definite at omega index {-st - 1}")
    return float(ec.value), e


def pw_to_grid(grid, g_pw, C_pw, pts=None):
    """Eq. 10: u[band][pt] = sum_Q C[band][Q] exp(+2 pi i Q.j/N) at the flat grid indices `pts` (default: all)."""
    grid, g_pw, C_pw = _i32(grid), _i32(g_pw).reshape(-1, 3), _c128(C_pw)
    C_pw = C_pw.reshape(-1, g_pw.shape[0])
    N = int(np.prod(grid))
    pts = np.arange(N, dtype=np.int64) if pts is None else np.ascontiguousarray(pts, dtype=np.int64)
    out = np.zeros((C_pw.shape[0], pts.size), dtype=np.complex128)
    lib().orc_pw_to_grid(_p(grid), C_pw.shape[0], g_pw.shape[0], _p(g_pw), _p(C_pw), pts.size, _p(pts), _p(out))
    return out


def symmetry_remap(grid, M, time_reversal, u):
    """Eq. 11: u_out(r) = u_in(M r) in reduced coordinates (M = T^-1, integer 3x3), conj if time_reversal."""
    grid, M, u = _i32(grid), _i32(M).reshape(9), _c128(u)
    N = int(np.prod(grid))
    out = np.empty_like(u)
    st = lib().orc_symmetry_remap(_p(grid), _p(M), int(bool(time_reversal)), u.size // N, _p(u), _p(out))
    if st != 0:
        raise ValueError("the symmetry operation does not map the grid onto itself")
    return out


def momentum_pw(cell, k_cart, g_pw, C_occ, C_unocc, n_proj=None, P_occ=None, P_unocc=None, Qgrad=None):
    """Eq. 15 / 19: grad[3][n_occ][n_unocc] = <psi_n| nabla |psi_m> from plane-wave coefficients (+ PAW term)."""
    g_pw = _i32(g_pw).reshape(-1, 3)
    C_occ, C_unocc = _c128(C_occ).reshape(-1, g_pw.shape[0]), _c128(C_unocc).reshape(-1, g_pw.shape[0])
    out = np.zeros((3, C_occ.shape[0], C_unocc.shape[0]), dtype=np.complex128)
    if n_proj is not None and len(n_proj):
        n_proj, P_occ, P_unocc, Qgrad = _i32(n_proj), _c128(P_occ), _c128(P_unocc), _c128(Qgrad)
        args = (n_proj.size, _p(n_proj), _p(P_occ), _p(P_unocc), _p(Qgrad))
    else:
        args = (0, None, None, None, None)
    lib().orc_momentum_pw(_p(_f64(cell).reshape(9)), _p(_f64(k_cart)), g_pw.shape[0], _p(g_pw), C_occ.shape[0], _p(C_occ),
                          C_unocc.shape[0], _p(C_unocc), *args, _p(out))
    return out


def optical_head(eps_occ, eps_unocc, qdir, grad):
    """Eq. 13: head[n][m] = -i qdir . grad[:, n, m] / (eps_m - eps_n)."""
    eo, eu, qd, grad = _f64(eps_occ), _f64(eps_unocc), _f64(qdir), _c128(grad)
    out = np.zeros((eo.size, eu.size), dtype=np.complex128)
    lib().orc_optical_head(eo.size, eu.size, _p(eo), _p(eu), _p(qd), _p(grad), _p(out))
    return out


class Chi0Oracle:
    """Same call shape as the library boundary (include/rpa_chi0.h), every step by the C oracle.

    ``g`` may be given explicitly (a sampled sub-list of the sphere): chi0 restricted to those G is exactly the
    chi0 of those G, because every element of Eq. 17 is an independent sum."""

    def __init__(self, grid, cell, q_red, ecut_ha, omega, omega_wt=None, g=None, mode="separable", spin_deg=None,
                 eta=None):
        """eta = None: omega are points i omega of the imaginary axis (the path).  eta > 0 (NEXT-4): omega are real
        frequencies and chi0 is evaluated at z = omega + i eta with the complex weights of ``weights_z``."""
        self.spin_deg = spin_deg
        self.eta = eta
        self.grid, self.cell, self.q = _i32(grid), _f64(cell).reshape(3, 3), _f64(q_red)
        self.omega = _f64(omega)
        self.omega_wt = None if omega_wt is None else _f64(omega_wt)
        if g is None:
            self.g, self.K2 = sphere(self.grid, self.cell, self.q, ecut_ha)
        else:
            self.g = _i32(g).reshape(-1, 3)
            self.K2 = K2_of(self.cell, self.q, self.g)
        self.ng = self.g.shape[0]
        self.mode = mode
        self.S = np.zeros((self.omega.size, self.ng, self.ng), dtype=np.complex128)
        self.n_pairs = 0

    def pair_densities(self, n, kd, n_proj=None, Q=None, R_cart=None):
        """n_nm(g) of occupied band index n (row of kd.psi_occ) against all kd.psi_unocc: [m][g]."""
        nt = pair_density(self.grid, kd.psi_occ[n], kd.psi_unocc, self.g, self.mode)
        if n_proj is not None and len(n_proj) > 0:
            paw_add(self.cell, self.q, self.g, n_proj, kd.P_occ[n], kd.P_unocc, Q, R_cart, nt)
        return nt

    def add_kpoint(self, kd, n_proj=None, Q=None, R_cart=None, head=None):
        """head[n][m] (optical limit, Eq. 13) replaces the G = 0 element of every pair density when given."""
        i0 = None
        if head is not None:
            i0 = int(np.flatnonzero((self.g == 0).all(axis=1))[0])
        for n in range(kd.psi_occ.shape[0]):
            nt = self.pair_densities(n, kd, n_proj, Q, R_cart)
            if head is not None:
                nt[:, i0] = head[n]
            if self.eta is None:
                w = weights(kd.eps_occ[n], kd.f_occ[n], kd.eps_unocc, kd.f_unocc, self.omega)
                accumulate(self.S, nt, w, kd.kweight)
            else:
                w = weights_z(kd.eps_occ[n], kd.f_occ[n], kd.eps_unocc, kd.f_unocc, self.omega + 1j * self.eta)
                accumulate_z(self.S, nt, w, kd.kweight)
            self.n_pairs += nt.shape[0]

    def get(self, i_omega=None):
        chi = chi0_from_S(self.S, volume(self.cell), self.spin_deg)
        return chi if i_omega is None else chi[i_omega]

    def ec_q(self, v):
        return ec_q(self.get(), v, self.omega_wt)
