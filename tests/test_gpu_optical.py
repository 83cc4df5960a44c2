"""Parity of the optical limit q -> 0 (Eq. 13, 15, 19; Table 1 step 10) against the CPU oracle,
through the C ABI: rpa_momentum_pw, rpa_chi0_add_kpoint_optical, rpa_ec_q with v(G = 0) = 4 pi."""
import numpy as np
import pytest

import oracle
from paper_1307_8052_b200 import workload as W
from tests.parity_util import rel_fro

pytestmark = pytest.mark.gpu


def _q0_config(seed=77):
    cell = np.array([[7.0, 0.2, 0.0], [0.0, 6.5, 0.3], [0.1, 0.0, 8.0]])
    return W.custom_config(seed, cell, (12, 10, 16), (0.0, 0.0, 0.0), n_occ=3, n_unocc=9, ng_target=40, n_omega=4, n_atoms=2,
                           n_proj_per_atom=3, orb_ecut_ha=3.0)


def _coeffs(cfg, bands):
    g = None
    C = []
    for b in bands:
        g, c = W.orbital_coefficients(cfg, 0, b)
        C.append(c)
    return g, np.stack(C)


def _qgrad(cfg, seed=5):
    rng = np.random.default_rng(seed)
    n = int((cfg.n_proj.astype(np.int64) ** 2).sum()) * 3
    return np.ascontiguousarray(rng.standard_normal(n) + 1j * rng.standard_normal(n))


def test_momentum_pw_matches_oracle():
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    g, Co = _coeffs(cfg, range(5))          # 5 "occupied": a ragged group of OPT_NB = 4
    _, Cu = _coeffs(cfg, range(5, 18))
    k = np.array([0.11, -0.2, 0.05])
    P = W.projections(cfg, 0)
    Qg = _qgrad(cfg)
    om, wt = W.omega_grid(cfg.n_omega)
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, int(cfg.n_proj.sum()), "cuda:0")
    try:
        a = B.rpa_momentum_pw(h, k, g, torch.from_numpy(Co).cuda(), torch.from_numpy(Cu).cuda()).cpu().numpy()
        b = B.rpa_momentum_pw(h, k, g, torch.from_numpy(Co).cuda(), torch.from_numpy(Cu).cuda(), cfg.n_proj,
                              torch.from_numpy(P[:5].copy()).cuda(), torch.from_numpy(P[5:18].copy()).cuda(),
                              torch.from_numpy(Qg).cuda()).cpu().numpy()
    finally:
        h.close()
    wa = oracle.momentum_pw(cfg.cell, k, g, Co, Cu)
    wb = oracle.momentum_pw(cfg.cell, k, g, Co, Cu, cfg.n_proj, P[:5], P[5:18], Qg)
    assert np.abs(a - wa).max() <= 1e-13 * np.abs(wa).max()
    assert np.abs(b - wb).max() <= 1e-13 * np.abs(wb).max()


def test_chi0_and_energy_in_the_optical_limit():
    """q = 0 handle: orbitals and gradients from plane-wave coefficients on the device, head replaced, chi0 and E_c(q)
    (v(G=0) = 4 pi) against the oracle; the plain add_kpoint must refuse a q = 0 handle."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = _q0_config()
    kd = W.kpoint(cfg, 0)
    g, Co = _coeffs(cfg, range(cfg.n_occ))
    _, Cu = _coeffs(cfg, range(cfg.n_occ, cfg.n_occ + cfg.n_unocc))
    kc = np.array([0.05, 0.1, -0.02])
    qdir = np.array([1.0, 2.0, -0.5])
    Qg = _qgrad(cfg)
    om, wt = W.omega_grid(cfg.n_omega)
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, int(cfg.n_proj.sum()), "cuda:0")
    try:
        gv, K2 = B.rpa_chi0_gvectors(h)
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).cuda()
        d = {k: torch.from_numpy(getattr(kd, k)).cuda() for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
        with pytest.raises(B.RpaError) as ei:
            B.rpa_chi0_add_kpoint(h, kd.kweight, d["psi_occ"], d["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc)
        assert ei.value.code == B.RPA_ERR_UNSUPPORTED
        grad = B.rpa_momentum_pw(h, kc, g, torch.from_numpy(Co).cuda(), torch.from_numpy(Cu).cuda(), cfg.n_proj, d["P_occ"],
                                 d["P_unocc"], torch.from_numpy(Qg).cuda())
        B.rpa_chi0_add_kpoint_optical(h, kd.kweight, d["psi_occ"], d["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ,
                                      kd.f_unocc, qdir, grad, cfg.n_proj, d["P_occ"], d["P_unocc"], Qd, W.atom_positions(cfg))
        chi = np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(cfg.n_omega)])
        i0 = int(np.flatnonzero((gv == 0).all(axis=1))[0])
        v = 4.0 * np.pi / np.where(K2 > 0, K2, 1.0)
        v[i0] = 4.0 * np.pi
        ec, e = B.rpa_ec_q(h, v)
    finally:
        h.close()
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    assert np.array_equal(orc.g, gv)
    gr = oracle.momentum_pw(cfg.cell, kc, g, Co, Cu, cfg.n_proj, kd.P_occ, kd.P_unocc, Qg)
    head = oracle.optical_head(kd.eps_occ, kd.eps_unocc, qdir / np.linalg.norm(qdir), gr)
    orc.add_kpoint(kd, cfg.n_proj, W.paw_Q(cfg, orc.K2), W.atom_positions(cfg), head=head)
    chi_o = orc.get()
    for i in range(cfg.n_omega):
        assert rel_fro(chi[i], chi_o[i]) <= 1e-10
        assert abs(chi[i][i0, i0] - chi_o[i][i0, i0]) <= 1e-12 * abs(chi_o[i][i0, i0])   # the head itself
    ec_o, e_o = orc.ec_q(v)
    assert abs(ec - ec_o) <= 1e-9 * abs(ec_o)


def test_optical_call_on_finite_q_handle_is_rejected():
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0, occ=[0], unocc=[0, 1])
    om, wt = W.omega_grid(cfg.n_omega)
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, 0, "cuda:0")
    try:
        grad = torch.zeros((3, 1, 2), dtype=torch.complex128, device="cuda")
        with pytest.raises(B.RpaError) as ei:
            B.rpa_chi0_add_kpoint_optical(h, 1.0, torch.from_numpy(kd.psi_occ).cuda(), torch.from_numpy(kd.psi_unocc).cuda(),
                                          kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc, [1.0, 0.0, 0.0], grad)
        assert ei.value.code == B.RPA_ERR_INVALID_ARG
    finally:
        h.close()


def test_real_axis_optical_limit():
    """The two NEXT rows together (the macroscopic dielectric function's ingredient): a q = 0 real-axis handle, head from
    the momentum matrix elements, chi0(omega + i eta) against the oracle's complex-weight route with the same head."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = _q0_config(seed=91)
    kd = W.kpoint(cfg, 0)
    g, Co = _coeffs(cfg, range(cfg.n_occ))
    _, Cu = _coeffs(cfg, range(cfg.n_occ, cfg.n_occ + cfg.n_unocc))
    kc = np.array([0.0, 0.0, 0.0])
    qdir = np.array([0.0, 0.0, 1.0])
    Qg = _qgrad(cfg, seed=9)
    om, eta = np.array([0.0, 0.4, 1.3]), 0.03
    h = B.rpa_chi0_create_real_axis(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, eta, 0, int(cfg.n_proj.sum()), "cuda:0")
    try:
        gv, K2 = B.rpa_chi0_gvectors(h)
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).cuda()
        d = {k: torch.from_numpy(getattr(kd, k)).cuda() for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
        grad = B.rpa_momentum_pw(h, kc, g, torch.from_numpy(Co).cuda(), torch.from_numpy(Cu).cuda(), cfg.n_proj, d["P_occ"],
                                 d["P_unocc"], torch.from_numpy(Qg).cuda())
        B.rpa_chi0_add_kpoint_optical(h, kd.kweight, d["psi_occ"], d["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ,
                                      kd.f_unocc, qdir, grad, cfg.n_proj, d["P_occ"], d["P_unocc"], Qd, W.atom_positions(cfg))
        chi = np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(len(om))])
    finally:
        h.close()
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, None, eta=eta)
    gr = oracle.momentum_pw(cfg.cell, kc, g, Co, Cu, cfg.n_proj, kd.P_occ, kd.P_unocc, Qg)
    head = oracle.optical_head(kd.eps_occ, kd.eps_unocc, qdir, gr)
    orc.add_kpoint(kd, cfg.n_proj, W.paw_Q(cfg, orc.K2), W.atom_positions(cfg), head=head)
    chi_o = orc.get()
    i0 = int(np.flatnonzero((gv == 0).all(axis=1))[0])
    for i in range(len(om)):
        assert rel_fro(chi[i], chi_o[i]) <= 1e-10
        assert abs(chi[i][i0, i0] - chi_o[i][i0, i0]) <= 1e-12 * abs(chi_o[i][i0, i0])
