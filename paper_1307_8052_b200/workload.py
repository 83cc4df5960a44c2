"""Seeded synthetic workloads shaped like the paper's systems (BASELINE.json configs[0..4]).

This module is the single source of inputs for BOTH the CPU oracle (``oracle/``) and the CUDA
library (``paper_1307_8052_b200.binding``).  It holds none of the method's arithmetic: it only
draws random numbers, builds orbitals from random plane-wave coefficients with a library inverse
FFT, and writes down cells, eigenvalues, occupations and frequency grids.  Anything indexed by the
G sphere (Q^a_ij(q+G), v_G) is generated from a ``K2 = |q+G|^2`` array that the *caller* obtains
from the side under test (oracle sphere or ``rpa_chi0_gvectors``), so no sphere logic of either
side leaks through here.

Recipe: DESIGN.md section 4; the paper's own inputs (P:L283-289,
Table 5: O2, Li2O, MoO3, N2/Ru(0001), CO/Ni(111) DFT orbitals) are not available, these stand in.
Units: Hartree atomic units (bohr, Ha).
"""
from __future__ import annotations

import dataclasses
from typing import Optional, Sequence

import numpy as np

HA_EV = 27.211386
ANG = 1.8897261  # bohr per angstrom
SEED0 = 13078052

_KIND_COEF, _KIND_EPS, _KIND_PROJ, _KIND_Q, _KIND_POS = 1, 2, 3, 4, 5


@dataclasses.dataclass(frozen=True)
class Config:
    index: int
    name: str
    cell: np.ndarray          # (3,3) rows a1,a2,a3 in bohr
    grid: tuple               # (N1,N2,N3)
    n_k: int
    q_red: tuple
    n_occ: int
    n_unocc: int
    ng_target: int
    n_omega: int
    n_atoms: int
    n_proj_per_atom: int
    gap_ev: Optional[float]   # None: no shift (cfg 0)
    smear_ev: Optional[float]  # None: f = 1/0
    orb_ecut_ha: float = 6.0

    @property
    def n_grid(self) -> int:
        return int(np.prod(self.grid))

    @property
    def n_pairs(self) -> int:
        return self.n_k * self.n_occ * self.n_unocc

    @property
    def n_proj(self) -> np.ndarray:
        return np.full(self.n_atoms, self.n_proj_per_atom, dtype=np.int32)

    @property
    def volume(self) -> float:
        return float(abs(np.linalg.det(self.cell)))


def _hex_cell(a_ang: float, c_ang: float) -> np.ndarray:
    a = a_ang * ANG
    return np.array([[a, 0.0, 0.0], [-0.5 * a, 0.5 * np.sqrt(3.0) * a, 0.0], [0.0, 0.0, c_ang * ANG]])


def _fcc_cell(a_ang: float) -> np.ndarray:
    h = 0.5 * a_ang * ANG
    return np.array([[0.0, h, h], [h, 0.0, h], [h, h, 0.0]])


CONFIGS = (
    Config(0, "toy", np.eye(3) * 8.0, (16, 16, 16), 1, (0.25, 0.0, 0.0), 4, 28, 150, 8, 2, 4, None, None),
    Config(1, "molecule", np.diag([12.0, 13.0, 14.0]) * ANG, (56, 60, 64), 1, (0.125, 0.0, 0.0),
           12, 600, 1200, 16, 2, 13, 5.0, None),
    Config(2, "bulk", _fcc_cell(4.6), (24, 24, 24), 64, (0.25, 0.0, 0.0), 8, 300, 400, 16, 3, 8, 5.0, None),
    Config(3, "slab", _hex_cell(5.4, 20.0), (40, 40, 168), 4, (0.5, 0.0, 0.0), 64, 1500, 3000, 16, 10, 18,
           None, 0.1),
    Config(4, "large_slab", _hex_cell(4.98, 23.0), (48, 48, 192), 8, (0.25, 0.25, 0.0), 120, 3000, 5000, 16,
           18, 18, None, 0.1),
)


def custom_config(index: int, cell, grid, q_red, n_occ, n_unocc, ng_target, n_omega, n_atoms, n_proj_per_atom,
                  n_k=1, gap_ev=None, smear_ev=None, orb_ecut_ha=6.0, name="custom") -> Config:
    """A test-sized config with the same recipe (used for tiny brute-force and ragged-tail cases)."""
    return Config(index, name, np.asarray(cell, dtype=np.float64), tuple(int(x) for x in grid), n_k,
                  tuple(float(x) for x in q_red), n_occ, n_unocc, ng_target, n_omega, n_atoms, n_proj_per_atom,
                  gap_ev, smear_ev, orb_ecut_ha)


def _rng(cfg: Config, kind: int, k: int = 0, band: int = 0) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([SEED0, cfg.index, kind, k, band]))


def recip(cell: np.ndarray) -> np.ndarray:
    """B = 2 pi A^-T, rows b_i with a_i . b_j = 2 pi delta_ij."""
    return 2.0 * np.pi * np.linalg.inv(np.asarray(cell, dtype=np.float64)).T


def tuned_ecut(cfg: Config) -> float:
    """E_cut (Ha) placed mid-way between two |q+G|^2/2 shells so that the sphere holds the first
    shell-complete count >= cfg.ng_target (the stated ~nG binds, not the stated Gcut).
    This is workload definition, not path arithmetic: it only picks a threshold with no float tie."""
    B = recip(cfg.cell)
    rng_ax = [np.arange(-((n - 1) // 2), (n - 1) // 2 + 1) for n in cfg.grid]
    g = np.stack(np.meshgrid(*rng_ax, indexing="ij"), axis=-1).reshape(-1, 3)
    K = (g + np.asarray(cfg.q_red)) @ B
    e = np.sort(0.5 * np.einsum("ij,ij->i", K, K))
    if cfg.ng_target > e.size:
        raise ValueError("ng_target exceeds the number of grid G vectors")
    e_star = e[cfg.ng_target - 1]
    tol = 1e-9 * max(e_star, 1.0)
    inside = e[e <= e_star + tol]
    outside = e[e > e_star + tol]
    if outside.size == 0:
        return float(inside[-1] * 1.01 + 1e-6)
    return float(0.5 * (inside[-1] + outside[0]))


def omega_grid(n_omega: int, omega0: float = 1.0):
    """Gauss-Legendre nodes mapped (-1,1)->(0,inf): w = w0 (1+x)/(1-x), weight 2 w0 c/(1-x)^2 (reading A11;
    the paper's own mapping, P:L50 'following Ref. [13]', is not in the container)."""
    x, c = np.polynomial.legendre.leggauss(n_omega)
    om = omega0 * (1.0 + x) / (1.0 - x)
    wt = 2.0 * omega0 * c / (1.0 - x) ** 2
    return np.ascontiguousarray(om), np.ascontiguousarray(wt)


def _coef_mask(cfg: Config):
    B = recip(cfg.cell)
    rng_ax = [np.fft.fftfreq(n, 1.0 / n).astype(np.int64) for n in cfg.grid]
    g = np.stack(np.meshgrid(*rng_ax, indexing="ij"), axis=-1)
    G = g @ B
    G2 = np.einsum("...i,...i->...", G, G)
    ok = 0.5 * G2 <= cfg.orb_ecut_ha
    for ax, n in enumerate(cfg.grid):
        ok &= np.abs(g[..., ax]) * 2 < n  # strict: Nyquist plane excluded
    return ok, np.exp(-G2 / 4.0)


class KPointData:
    """All arrays the boundary call ``rpa_chi0_add_kpoint`` takes for one k-point (host, numpy)."""

    def __init__(self, cfg, k, psi_occ, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc, P_occ, P_unocc):
        self.cfg, self.k = cfg, k
        self.psi_occ, self.psi_unocc = psi_occ, psi_unocc
        self.eps_occ, self.eps_unocc = eps_occ, eps_unocc
        self.f_occ, self.f_unocc = f_occ, f_unocc
        self.P_occ, self.P_unocc = P_occ, P_unocc
        self.kweight = 1.0 / cfg.n_k


def orbital(cfg: Config, k: int, band: int, _cache={}) -> np.ndarray:
    """Periodic part u(r_j) of band `band` at k-point `k`: seeded Gaussian plane-wave coefficients with
    decay exp(-|G|^2/4) inside |G|^2/2 <= 6 Ha, inverse FFT, grid-normalised: (1/N) sum |u|^2 = 1."""
    key = (cfg.index, cfg.grid, cfg.orb_ecut_ha, cfg.cell.tobytes())
    if key not in _cache:
        _cache.clear()
        _cache[key] = _coef_mask(cfg)
    ok, decay = _cache[key]
    r = _rng(cfg, _KIND_COEF, k, band)
    nsel = int(ok.sum())
    xi = r.standard_normal((nsel, 2))
    C = np.zeros(cfg.grid, dtype=np.complex128)
    C[ok] = (xi[:, 0] + 1j * xi[:, 1]) * decay[ok]
    u = np.fft.ifftn(C) * cfg.n_grid
    u *= 1.0 / np.sqrt(np.mean(np.abs(u) ** 2))
    return np.ascontiguousarray(u)


def orbital_coefficients(cfg: Config, k: int, band: int, _mask=None):
    """(g_pw[n_pw][3] int32, C[n_pw]): the plane-wave coefficients behind `orbital`, scaled so that sum |C|^2 = 1
    (Parseval: the grid orbital sum_Q C(Q) exp(2 pi i Q.j/N) is then grid-normalised).  Same random stream as
    `orbital`, so pw -> grid of these coefficients reproduces it to rounding."""
    if _mask is None:   # (ok, decay[ok], g[ok]): the same for every band of a config
        ok, decay = _coef_mask(cfg)
        rng_ax = [np.fft.fftfreq(n, 1.0 / n).astype(np.int64) for n in cfg.grid]
        g = np.stack(np.meshgrid(*rng_ax, indexing="ij"), axis=-1)
        _mask = (ok, decay[ok], np.ascontiguousarray(g[ok].astype(np.int32)))
    ok, dec, gsel = _mask
    xi = _rng(cfg, _KIND_COEF, k, band).standard_normal((dec.size, 2))
    C = (xi[:, 0] + 1j * xi[:, 1]) * dec
    C *= 1.0 / np.sqrt(np.sum(np.abs(C) ** 2))
    return gsel, np.ascontiguousarray(C)


def kpoint_coefficients(cfg: Config, k: int, occ: Optional[Sequence[int]] = None,
                        unocc: Optional[Sequence[int]] = None):
    """(g_pw, C_occ[n_occ][n_pw], C_unocc[n_unocc][n_pw]): the plane-wave form of `kpoint`'s orbitals (same bands,
    same random streams; all bands share one coefficient sphere)."""
    occ = range(cfg.n_occ) if occ is None else occ
    unocc = range(cfg.n_unocc) if unocc is None else unocc
    ok, decay = _coef_mask(cfg)
    rng_ax = [np.fft.fftfreq(n, 1.0 / n).astype(np.int64) for n in cfg.grid]
    g = np.stack(np.meshgrid(*rng_ax, indexing="ij"), axis=-1)
    mask = (ok, decay[ok], np.ascontiguousarray(g[ok].astype(np.int32)))
    out = []
    for bands in ([int(b) for b in occ], [cfg.n_occ + int(b) for b in unocc]):
        rows = [orbital_coefficients(cfg, k, b, mask)[1] for b in bands]
        out.append(np.ascontiguousarray(np.stack(rows)) if rows else np.zeros((0, mask[1].size), dtype=np.complex128))
    return mask[2], out[0], out[1]


def eigenvalues(cfg: Config, k: int):
    """eps (Ha) sorted, occupations per spin channel in [0,1]."""
    nb = cfg.n_occ + cfg.n_unocc
    eps = np.sort(_rng(cfg, _KIND_EPS, k).uniform(-1.0, 1.0, nb))
    if cfg.gap_ev is not None:
        gap = cfg.gap_ev / HA_EV
        eps[cfg.n_occ:] += gap - (eps[cfg.n_occ] - eps[cfg.n_occ - 1])
    if cfg.smear_ev is None:
        f = np.concatenate([np.ones(cfg.n_occ), np.zeros(cfg.n_unocc)])
    else:
        kt = cfg.smear_ev / HA_EV
        mu = 0.5 * (eps[cfg.n_occ - 1] + eps[cfg.n_occ])
        x = np.clip((eps - mu) / kt, -700.0, 700.0)
        f = 1.0 / (1.0 + np.exp(x))
    return eps, f


def projections(cfg: Config, k: int) -> np.ndarray:
    """P[band][sum_a n_proj] ~ N(0,0.1) + i N(0,0.1)."""
    nb = cfg.n_occ + cfg.n_unocc
    ntot = int(cfg.n_proj.sum())
    x = _rng(cfg, _KIND_PROJ, k).standard_normal((nb, ntot, 2)) * 0.1
    return np.ascontiguousarray(x[..., 0] + 1j * x[..., 1])


def kpoint(cfg: Config, k: int, occ: Optional[Sequence[int]] = None,
           unocc: Optional[Sequence[int]] = None) -> KPointData:
    """Arrays of k-point `k`; `occ` / `unocc` pick band slices (indices within the occupied / unoccupied
    sets), default all.  Any band regenerates alone, so slices equal the corresponding rows of a full run."""
    occ = list(range(cfg.n_occ)) if occ is None else [int(i) for i in occ]
    unocc = list(range(cfg.n_unocc)) if unocc is None else [int(i) for i in unocc]
    eps, f = eigenvalues(cfg, k)
    P = projections(cfg, k)
    bo = np.asarray(occ, dtype=np.int64)
    bu = np.asarray(unocc, dtype=np.int64) + cfg.n_occ
    psi_occ = np.empty((len(occ),) + tuple(cfg.grid), dtype=np.complex128)
    psi_unocc = np.empty((len(unocc),) + tuple(cfg.grid), dtype=np.complex128)
    for i, b in enumerate(bo):
        psi_occ[i] = orbital(cfg, k, int(b))
    for i, b in enumerate(bu):
        psi_unocc[i] = orbital(cfg, k, int(b))
    c = np.ascontiguousarray
    return KPointData(cfg, k, psi_occ, psi_unocc, c(eps[bo]), c(eps[bu]), c(f[bo]), c(f[bu]), c(P[bo]), c(P[bu]))


def atom_positions(cfg: Config) -> np.ndarray:
    """R_a in Cartesian bohr, fractional coordinates uniform[0,1)^3."""
    frac = _rng(cfg, _KIND_POS).uniform(0.0, 1.0, (cfg.n_atoms, 3))
    return np.ascontiguousarray(frac @ cfg.cell)


def paw_Q(cfg: Config, K2: np.ndarray) -> np.ndarray:
    """Q[a][i][j][g], atoms concatenated (flat complex128): Hermitian in (i,j) for every g,
    seeded Gaussians x exp(-|q+G|^2/8) (BASELINE.json configs[0]).  K2[g] = |q+G_g|^2 in the caller's order."""
    K2 = np.asarray(K2, dtype=np.float64)
    ng = K2.size
    out = []
    for a in range(cfg.n_atoms):
        ni = int(cfg.n_proj[a])
        r = _rng(cfg, _KIND_Q, a)
        X = r.standard_normal((ni, ni, ng, 2))
        X = X[..., 0] + 1j * X[..., 1]
        Qa = 0.5 * (X + np.conj(np.swapaxes(X, 0, 1))) * np.exp(-K2 / 8.0)
        out.append(Qa.reshape(-1))
    if not out:
        return np.zeros(0, dtype=np.complex128)
    return np.ascontiguousarray(np.concatenate(out))


def coulomb(K2: np.ndarray) -> np.ndarray:
    """v_G(q) = 4 pi / |q+G|^2."""
    return 4.0 * np.pi / np.asarray(K2, dtype=np.float64)


def plane_wave_orbitals(grid, gvecs) -> np.ndarray:
    """u_b(j) = exp(2 pi i g_b . j / N) for the closed-form (discrete Lindhard) checks."""
    N1, N2, N3 = grid
    j1 = np.arange(N1)[:, None, None] / N1
    j2 = np.arange(N2)[None, :, None] / N2
    j3 = np.arange(N3)[None, None, :] / N3
    out = np.empty((len(gvecs), N1, N2, N3), dtype=np.complex128)
    for b, g in enumerate(gvecs):
        out[b] = np.exp(2j * np.pi * (g[0] * j1 + g[1] * j2 + g[2] * j3))
    return out
