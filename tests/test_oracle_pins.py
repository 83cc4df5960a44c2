"""Pins of the CPU oracle (oracle/rpa_oracle.c) against what the paper and the mathematics fix.

The paper prints no numeric chi0 or E_c, so every pin is a closed form, a library
special case, brute force on a tiny grid, or an invariant.  Each test names
the oracle routine it pins and the mistake it would catch.  CPU only.
"""
import types

import numpy as np
import pytest

import oracle
from paper_1307_8052_b200 import workload as W


def _flat_index(g, grid):
    g = np.asarray(g)
    return ((g[:, 0] % grid[0]) * grid[1] + (g[:, 1] % grid[1])) * grid[2] + (g[:, 2] % grid[2])


def _kd(cfg, psi_occ, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc, P_occ=None, P_unocc=None, kweight=1.0):
    c = np.ascontiguousarray
    return types.SimpleNamespace(cfg=cfg, psi_occ=c(psi_occ), psi_unocc=c(psi_unocc), eps_occ=c(eps_occ),
                                 eps_unocc=c(eps_unocc), f_occ=c(f_occ), f_unocc=c(f_unocc), P_occ=P_occ,
                                 P_unocc=P_unocc, kweight=kweight)


# ---------------------------------------------------------------- sphere (orc_sphere, orc_K2, orc_volume)
def test_sphere_matches_bruteforce_enumeration(tiny_cfg):
    """Pins orc_sphere: membership, strict Nyquist exclusion, ordering (A6, A7) and B = 2 pi A^-T."""
    cfg = tiny_cfg
    ecut = W.tuned_ecut(cfg)
    g, K2 = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, ecut)
    B = 2 * np.pi * np.linalg.inv(cfg.cell).T
    assert np.allclose(cfg.cell @ B.T, 2 * np.pi * np.eye(3), atol=1e-13)
    want = []
    for a in range(-cfg.grid[0], cfg.grid[0] + 1):
        for b in range(-cfg.grid[1], cfg.grid[1] + 1):
            for c in range(-cfg.grid[2], cfg.grid[2] + 1):
                if 2 * abs(a) >= cfg.grid[0] or 2 * abs(b) >= cfg.grid[1] or 2 * abs(c) >= cfg.grid[2]:
                    continue
                K = (np.array([a, b, c]) + np.array(cfg.q_red)) @ B
                if 0.5 * K @ K <= ecut:
                    want.append((a, b, c))
    want = np.array(want)
    want = want[np.argsort(_flat_index(want, cfg.grid))]
    assert g.shape == want.shape and (g == want).all()
    assert len(g) >= cfg.ng_target
    K = (g + np.array(cfg.q_red)) @ B
    assert np.allclose(K2, np.einsum("ij,ij->i", K, K), rtol=1e-14)
    assert np.allclose(oracle.K2_of(cfg.cell, cfg.q_red, g[::3]), K2[::3], rtol=1e-15)
    assert np.isclose(oracle.volume(cfg.cell), abs(np.linalg.det(cfg.cell)), rtol=1e-14)


def test_sphere_sizes_of_the_five_configs():
    """The tuned cut-offs give the ~nG of BASELINE.json configs (A18) -- guards the workload definition."""
    want = {0: 155, 1: 1200, 2: 401, 3: 3004, 4: 5001}
    for cfg in W.CONFIGS:
        g, _ = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
        assert len(g) == want[cfg.index]
        assert (np.diff(_flat_index(g, cfg.grid)) > 0).all()


# ---------------------------------------------------------------- pair density (P1, P2, P3)
def test_pair_density_bruteforce_einsum(tiny_cfg):
    """P1: naive == separable == a numpy einsum of Eq. 7 (sign of the exponent, 1/N, conj on u_n, axis order)."""
    cfg = tiny_cfg
    g, _ = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
    kd = W.kpoint(cfg, 0)
    N1, N2, N3 = cfg.grid
    j1, j2, j3 = np.arange(N1), np.arange(N2), np.arange(N3)
    E1 = np.exp(-2j * np.pi * np.outer(g[:, 0], j1) / N1)
    E2 = np.exp(-2j * np.pi * np.outer(g[:, 1], j2) / N2)
    E3 = np.exp(-2j * np.pi * np.outer(g[:, 2], j3) / N3)
    for n in range(cfg.n_occ):
        prod = np.conj(kd.psi_occ[n])[None] * kd.psi_unocc
        want = np.einsum("mabc,ga,gb,gc->mg", prod, E1, E2, E3) / cfg.n_grid
        nv = oracle.pair_density(cfg.grid, kd.psi_occ[n], kd.psi_unocc, g, "naive")
        sp = oracle.pair_density(cfg.grid, kd.psi_occ[n], kd.psi_unocc, g, "separable")
        scale = np.abs(want).max()
        assert np.abs(nv - want).max() <= 1e-14 * max(scale, 1)
        assert np.abs(sp - want).max() <= 1e-14 * max(scale, 1)


def test_pair_density_is_gathered_library_fft():
    """P2: ntilde = gather(numpy.fft.fftn(conj(u_n) u_m)) / N on config 0 (library special case)."""
    cfg = W.CONFIGS[0]
    g, _ = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
    kd = W.kpoint(cfg, 0, occ=[1], unocc=[0, 5, 27])
    got = oracle.pair_density(cfg.grid, kd.psi_occ[0], kd.psi_unocc, g, "separable")
    idx = _flat_index(g, cfg.grid)
    for m in range(3):
        F = np.fft.fftn(np.conj(kd.psi_occ[0]) * kd.psi_unocc[m]).reshape(-1) / cfg.n_grid
        assert np.abs(got[m] - F[idx]).max() <= 1e-14
    nv = oracle.pair_density(cfg.grid, kd.psi_occ[0], kd.psi_unocc[:1], g[::7], "naive")
    assert np.abs(nv[0] - got[0, ::7]).max() <= 1e-14


def test_normalisation_n_nn_is_one():
    """P3: q = 0, G = 0 => n_nn = <psi_n|psi_n> = 1 for grid-normalised orbitals; delta_nm for
    orthonormal plane waves."""
    cfg = W.CONFIGS[0]
    u = W.orbital(cfg, 0, 2)
    g0 = np.zeros((1, 3), dtype=np.int32)
    n = oracle.pair_density(cfg.grid, u, u[None], g0)
    assert abs(n[0, 0] - 1.0) <= 1e-14
    pw = W.plane_wave_orbitals(cfg.grid, [(0, 0, 0), (1, 0, -1), (2, 1, 0)])
    for a in range(3):
        n = oracle.pair_density(cfg.grid, pw[a], pw, g0, "naive")[:, 0]
        assert np.abs(n - np.eye(3)[a]).max() <= 1e-14


# ---------------------------------------------------------------- weights (Eq. 18, A1)
def test_weights_are_twice_real_part_of_eq18():
    """Pins orc_weights: w = 2 Re[(f_n - f_m)/(i w + eps_n - eps_m)] (Eq. 18 without 2/Omega)."""
    rng = np.random.default_rng(5)
    eps_m, f_m = rng.uniform(-1, 1, 7), rng.uniform(0, 1, 7)
    om = np.array([0.05, 1.0, 30.0])
    w = oracle.weights(-0.3, 0.9, eps_m, f_m, om)
    want = 2 * np.real((0.9 - f_m)[None, :] / (1j * om[:, None] + (-0.3 - eps_m)[None, :]))
    assert np.allclose(w, want, rtol=1e-14, atol=0)
    # eps_n == eps_m => w = 0 (A12)
    assert oracle.weights(0.2, 1.0, np.array([0.2]), np.array([0.0]), om).max() == 0.0


# ---------------------------------------------------------------- accumulate (P6, P7, P8)
def test_constant_weight_case_is_library_NNH(tiny_cfg):
    """P8: eps_occ = -1/2, eps_unocc = +1/2, f = 1/0 => chi0 = -(2 s/Omega)/(w^2+1) N N^H (library matmul)."""
    cfg = tiny_cfg
    kd = W.kpoint(cfg, 0)
    om = np.array([0.3, 2.0])
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om)
    kd.eps_occ[:] = -0.5
    kd.eps_unocc[:] = 0.5
    Ns = []
    for n in range(cfg.n_occ):
        Ns.append(orc.pair_densities(n, kd))
    orc.add_kpoint(kd)
    Nmat = np.concatenate(Ns, 0).T  # [g][pair]
    for i, w in enumerate(om):
        want = -(2 * 2 / cfg.volume) / (w * w + 1) * (Nmat @ Nmat.conj().T)
        got = orc.get(i)
        assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want)


def test_hermitian_and_negative_semidefinite():
    """P6, P7 on config 0 (f = 1/0) and with smeared occupations (A12): both triangles are filled
    independently, so Hermiticity is a real check; chi0(i w) is negative semidefinite."""
    cfg = W.CONFIGS[0]
    om, wt = W.omega_grid(3)
    g, K2 = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
    gs = g[::3]
    kd = W.kpoint(cfg, 0, unocc=range(0, 28, 3))
    for smear in (False, True):
        if smear:
            mu = 0.5 * (kd.eps_occ[-1] + kd.eps_unocc[0])
            kd.f_occ = 1 / (1 + np.exp((kd.eps_occ - mu) / 0.05))
            kd.f_unocc = 1 / (1 + np.exp((kd.eps_unocc - mu) / 0.05))
        orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, 0.0, om, g=gs)
        orc.add_kpoint(kd)
        chi = orc.get()
        for i in range(3):
            nrm = np.linalg.norm(chi[i])
            assert nrm > 0
            assert np.linalg.norm(chi[i] - chi[i].conj().T) <= 1e-14 * nrm
            assert np.linalg.eigvalsh(0.5 * (chi[i] + chi[i].conj().T)).max() <= 1e-13 * nrm


# ---------------------------------------------------------------- closed forms for the whole chain (P4, P5)
def _lindhard_setup():
    grid = (8, 6, 10)
    cell = np.array([[6.0, 0.0, 0.0], [0.5, 5.0, 0.0], [0.0, 0.3, 7.0]])
    cfg = W.custom_config(101, cell, grid, (0.25, 0.0, 0.5), 0, 0, 30, 3, 0, 0)
    g_occ = [(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 1), (0, -1, -1)]  # inversion symmetric
    g_unocc = [(2, 0, 0), (1, 1, 0), (0, 0, 2), (-1, 1, 1), (0, 1, 2), (1, 0, 1), (2, 0, 1), (0, 0, 1), (1, 1, 2),
               (-1, -1, 0), (0, -1, 0), (-2, 0, 1), (-1, 0, 1)]
    return cfg, g_occ, g_unocc


def test_plane_wave_orbitals_give_discrete_lindhard_sum():
    """P4: u_n = exp(2 pi i g_n.j/N) => ntilde_nm(g) = delta(g, g_m - g_n); chi0 is exactly diagonal with
    chi0_gg = (2/Omega) sum_k wk sum_{g_m - g_n = g} w_nm(w), eps = |(k+g)B|^2/2.  Catches a wrong sign in the
    exponent, transposed g/g', a dropped prefactor, a wrong weight, wrong G ordering."""
    cfg, g_occ, g_unocc = _lindhard_setup()
    B = W.recip(cfg.cell)
    om = np.array([0.2, 1.5, 9.0])
    ecut = W.tuned_ecut(cfg)
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, ecut, om, mode="naive")
    ks = [np.array([0.0, 0.0, 0.0]), np.array([0.5, 0.25, 0.0])]
    want = np.zeros((3, orc.ng))
    where = {tuple(int(x) for x in gg): i for i, gg in enumerate(orc.g)}
    pw_o = W.plane_wave_orbitals(cfg.grid, g_occ)
    pw_u = W.plane_wave_orbitals(cfg.grid, g_unocc)
    for k in ks:
        eo = np.array([0.5 * np.sum(((k + np.array(x)) @ B) ** 2) for x in g_occ])
        eu = np.array([0.5 * np.sum(((k + np.array(cfg.q_red) + np.array(x)) @ B) ** 2) for x in g_unocc])
        kd = _kd(cfg, pw_o, pw_u, eo, eu, np.ones(len(g_occ)), np.zeros(len(g_unocc)), kweight=0.5)
        orc.add_kpoint(kd)
        for a, gn in enumerate(g_occ):
            for b, gm in enumerate(g_unocc):
                d = tuple(np.array(gm) - np.array(gn))
                if d in where:
                    de = eo[a] - eu[b]
                    want[:, where[d]] += 0.5 * (2 / cfg.volume) * 2 * de / (om ** 2 + de ** 2)
    chi = orc.get()
    assert np.count_nonzero(want[0]) >= 10
    for i in range(3):
        assert np.abs(chi[i] - np.diag(np.diag(chi[i]))).max() <= 1e-15
        assert np.abs(np.diag(chi[i]).imag).max() <= 1e-16
        assert np.allclose(np.diag(chi[i]).real, want[i], rtol=1e-13, atol=1e-17)


def test_f_sum_rule():
    """P5 (textbook): w^2 chi0_gg(i w) -> -n_e |q+G|^2, n_e = 2 N_occ/Omega, for w -> inf.  It comes out only
    with BOTH factors of 2 (spin in 2/Omega and the 2 Re of A1) -- pins the prefactor readings A1-A3."""
    cfg, g_occ, _ = _lindhard_setup()
    B = W.recip(cfg.cell)
    gsel = np.array([[2, 1, 3]], dtype=np.int32)  # g_n + g is unoccupied for every n
    g_unocc = [tuple(np.array(x) + gsel[0]) for x in g_occ]
    om = np.array([1.0e4])
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, 0.0, om, g=gsel, mode="naive")
    eo = np.array([0.5 * np.sum((np.array(x) @ B) ** 2) for x in g_occ])
    eu = np.array([0.5 * np.sum(((np.array(cfg.q_red) + np.array(x)) @ B) ** 2) for x in g_unocc])
    kd = _kd(cfg, W.plane_wave_orbitals(cfg.grid, g_occ), W.plane_wave_orbitals(cfg.grid, g_unocc), eo, eu,
             np.ones(5), np.zeros(5))
    orc.add_kpoint(kd)
    n_e = 2 * len(g_occ) / cfg.volume
    ratio = (om[0] ** 2 * orc.get(0)[0, 0].real) / (-n_e * orc.K2[0])
    assert abs(ratio - 1) < 1e-6


# ---------------------------------------------------------------- PAW (P9)
def test_paw_single_projector_closed_form(tiny_cfg):
    """P9a: one atom, one projector: dn_nm(g) = conj(p_n) p_m c_g exp(-i K_g.R) (sign of the phase, conj on P_n)."""
    cfg = tiny_cfg
    g, K2 = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
    B = W.recip(cfg.cell)
    rng = np.random.default_rng(3)
    R = np.array([[0.7, -1.1, 2.3]])
    c = rng.standard_normal(len(g)) + 1j * rng.standard_normal(len(g))
    p_n = np.array([0.3 - 0.8j])
    p_m = (rng.standard_normal((4, 1)) + 1j * rng.standard_normal((4, 1)))
    n = np.zeros((4, len(g)), dtype=np.complex128)
    oracle.paw_add(cfg.cell, cfg.q_red, g, [1], p_n, p_m, c, R, n)
    K = (g + np.array(cfg.q_red)) @ B
    want = np.conj(p_n[0]) * p_m[:, :1] * (c * np.exp(-1j * K @ R[0]))[None, :]
    assert np.abs(n - want).max() <= 1e-14 * np.abs(want).max()


def test_paw_random_ragged_vs_einsum(tiny_cfg):
    """P9b: two atoms with 3 and 2 projectors, non-Hermitian Q (A10: no symmetry assumed), vs numpy einsum;
    and the reassociated form T_n = conj(P_n) Q first (what the GPU does) equals the direct form."""
    cfg = tiny_cfg
    g, _ = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
    ng = len(g)
    B = W.recip(cfg.cell)
    rng = np.random.default_rng(4)
    n_proj = [3, 2]
    R = rng.uniform(-3, 3, (2, 3))
    cplx = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    Qa = [cplx(3, 3, ng), cplx(2, 2, ng)]
    Q = np.concatenate([q.reshape(-1) for q in Qa])
    P_n, P_m = cplx(5), cplx(4, 5)
    base = cplx(4, ng)
    n = base.copy()
    oracle.paw_add(cfg.cell, cfg.q_red, g, n_proj, P_n, P_m, Q, R, n)
    K = (g + np.array(cfg.q_red)) @ B
    want = base.copy()
    off = 0
    for a, ni in enumerate(n_proj):
        ph = np.exp(-1j * K @ R[a])
        want += np.einsum("i,ijg,mj,g->mg", np.conj(P_n[off:off + ni]), Qa[a], P_m[:, off:off + ni], ph)
        T = np.einsum("i,ijg->jg", np.conj(P_n[off:off + ni]), Qa[a]) * ph
        assert np.allclose(np.einsum("jg,mj->mg", T, P_m[:, off:off + ni]),
                           np.einsum("i,ijg,mj,g->mg", np.conj(P_n[off:off + ni]), Qa[a], P_m[:, off:off + ni], ph),
                           rtol=1e-13)
        off += ni
    assert np.abs(n - want).max() <= 1e-13 * np.abs(want).max()


# ---------------------------------------------------------------- invariants of the whole chain (P10)
def _full_chi(cfg, kds, om, n_proj=None, Q=None, R=None):
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om)
    for kd in kds:
        orc.add_kpoint(kd, n_proj, Q, R)
    return orc


def test_gauge_permutation_additivity(tiny_cfg):
    """P10: u_n -> e^{i t} u_n with P_n -> e^{i t} P_n leaves chi0 unchanged; permuting bands (with eps, f, P)
    leaves it unchanged; splitting bands over calls leaves it unchanged."""
    cfg = tiny_cfg
    om = np.array([0.4, 3.0])
    _, K2 = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
    Q, R = W.paw_Q(cfg, K2), W.atom_positions(cfg)
    kd = W.kpoint(cfg, 0)
    ref = _full_chi(cfg, [kd], om, cfg.n_proj, Q, R).get()
    nrm = np.linalg.norm(ref)
    # gauge
    rng = np.random.default_rng(9)
    kg = W.kpoint(cfg, 0)
    for arr_psi, arr_P in ((kg.psi_occ, kg.P_occ), (kg.psi_unocc, kg.P_unocc)):
        for b in range(arr_psi.shape[0]):
            ph = np.exp(1j * rng.uniform(0, 2 * np.pi))
            arr_psi[b] *= ph
            arr_P[b] *= ph
    assert np.linalg.norm(_full_chi(cfg, [kg], om, cfg.n_proj, Q, R).get() - ref) <= 1e-13 * nrm
    # permutation of the unoccupied bands
    perm = rng.permutation(cfg.n_unocc)
    kp = W.kpoint(cfg, 0, unocc=perm)
    assert np.linalg.norm(_full_chi(cfg, [kp], om, cfg.n_proj, Q, R).get() - ref) <= 1e-13 * nrm
    # additivity over band splits
    parts = [W.kpoint(cfg, 0, occ=[0], unocc=[0, 1, 2]), W.kpoint(cfg, 0, occ=[0], unocc=[3, 4]),
             W.kpoint(cfg, 0, occ=[1])]
    assert np.linalg.norm(_full_chi(cfg, parts, om, cfg.n_proj, Q, R).get() - ref) <= 1e-13 * nrm
    # the PAW term matters in this test (guards against a silently dropped correction)
    assert np.linalg.norm(_full_chi(cfg, [kd], om).get() - ref) > 1e-3 * nrm


# ---------------------------------------------------------------- energy (P11, P12)
def test_ec_routes_agree():
    """P11: Cholesky log-det route == sum_i [ln(1 - l_i) + l_i] with l = eigvalsh(D chi D) == eigenvalues of the
    non-symmetric v chi (A14); diagonal chi => per-G closed form; small-X limit e ~ -Tr X^2 / 2."""
    rng = np.random.default_rng(11)
    ng, nw = 24, 3
    chi = np.zeros((nw, ng, ng), dtype=np.complex128)
    for i in range(nw):
        A = rng.standard_normal((ng, 40)) + 1j * rng.standard_normal((ng, 40))
        chi[i] = -(A @ A.conj().T) * 0.02 / (i + 1)
    v = rng.uniform(0.5, 20.0, ng)
    wt = np.array([0.3, 1.1, 2.5])
    ec, e = oracle.ec_q(chi, v, wt)
    D = np.sqrt(v)
    for i in range(nw):
        lam = np.linalg.eigvalsh(D[:, None] * chi[i] * D[None, :])
        assert np.isclose(e[i], np.sum(np.log1p(-lam) + lam), rtol=1e-12)
        lam2 = np.linalg.eigvals(v[:, None] * chi[i])
        assert np.isclose(e[i], np.sum(np.log(1 - lam2) + lam2).real, rtol=1e-11)
    assert np.isclose(ec, (wt @ e) / (2 * np.pi), rtol=1e-14)
    d = -rng.uniform(0.01, 0.5, ng)
    chid = np.stack([np.diag(d).astype(np.complex128)] * nw)
    _, ed = oracle.ec_q(chid, v, wt)
    assert np.allclose(ed, np.sum(np.log(1 - v * d) + v * d), rtol=1e-13)
    small = chi[:1] * 1e-4
    _, es = oracle.ec_q(small, v, wt[:1])
    X = D[:, None] * small[0] * D[None, :]
    assert np.isclose(es[0], -0.5 * np.trace(X @ X).real, rtol=1e-2)
    with pytest.raises(FloatingPointError):
        oracle.ec_q(-chi * 1e4, v, wt)  # positive chi => I - X indefinite


def test_frequency_quadrature():
    """P12 (harness, A11): sum wt_i h(w_i) for h = 1/(1+w^2)^2 equals pi/4."""
    om, wt = W.omega_grid(16)
    assert abs(np.sum(wt / (1 + om ** 2) ** 2) - np.pi / 4) < 1e-10
    assert (om > 0).all() and (wt > 0).all()


# ---------------------------------------------------------------- stored values written by the oracle
def test_golden_toy_values():
    """tests/golden/toy_oracle.txt is written by tests/golden/make_golden.py, which calls only oracle/;
    this guards the oracle's arithmetic against silent edits (a change must cite its justification)."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "toy_oracle.txt")
    from tests.golden.make_golden import compute
    vals = compute()
    want = {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        k, re, im = line.split()
        want[k] = complex(float(re), float(im))
    assert set(want) == set(vals)
    for k in want:
        assert abs(vals[k] - want[k]) <= 1e-12 * max(1e-300, abs(want[k])), k


def test_explicit_spin_channels_equal_the_spin_paired_sum():
    """NEXT-4: two identical spin channels summed with s = 1 give the spin-paired chi0 (s = 2, reading A3)."""
    cfg = W.custom_config(55, np.diag([6.0, 6.5, 7.0]), (6, 6, 6), (0.25, 0.0, 0.0), n_occ=2, n_unocc=4, ng_target=8,
                          n_omega=3, n_atoms=1, n_proj_per_atom=2, orb_ecut_ha=2.0)
    kd = W.kpoint(cfg, 0)
    om, wt = W.omega_grid(cfg.n_omega)
    paired = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    paired.add_kpoint(kd)
    spin = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, spin_deg=1)
    spin.add_kpoint(kd)
    spin.add_kpoint(kd)   # the second channel
    assert np.abs(spin.get() - paired.get()).max() <= 1e-15 * np.abs(paired.get()).max()
