"""SURVEY 8(f) NEXT-4, second workload: chi0 on the real frequency axis (rpa_chi0_create_real_axis) against the
oracle's complex-weight route (orc_weights_z / orc_accumulate_z), element by element; through the C ABI."""
import numpy as np
import pytest

from paper_1307_8052_b200 import workload as W
from tests.parity_util import gpu_run, oracle_run, rel_fro

pytestmark = pytest.mark.gpu

CHI_TOL = 1e-10
OMEGA = np.array([0.0, 0.11, 0.5, -0.5, 2.0, 40.0])
ETA = 0.05


def _gpu_real_axis(cfg, kds, omega, eta, use_paw=True, batch=0, device_resident=False):
    import torch
    from paper_1307_8052_b200 import binding as B
    ptot = int(cfg.n_proj.sum()) if use_paw else 0
    h = B.rpa_chi0_create_real_axis(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), omega, eta, batch, ptot, "cuda:0")
    try:
        g, K2 = B.rpa_chi0_gvectors(h)
        Qd = R = npj = None
        if ptot:
            Qd, R, npj = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0"), W.atom_positions(cfg), cfg.n_proj
        for kd in kds:
            if device_resident:
                dv = {k: torch.from_numpy(getattr(kd, k)).to("cuda:0") for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
                B.rpa_chi0_add_kpoint(h, kd.kweight, dv["psi_occ"], dv["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ,
                                      kd.f_unocc, npj, dv["P_occ"] if ptot else None, dv["P_unocc"] if ptot else None, Qd, R)
                B.rpa_chi0_sync(h)
            else:
                B.add_kpoint_host(h, kd, npj, Qd, R)
        yield h, g, K2
    finally:
        h.close()


def test_config0_real_axis_full():
    """Toy config, all bands, PAW on: every element of chi0(omega + i eta) for positive, negative, zero and far
    off-resonance frequencies; the adjoint relation chi0(-omega) = chi0(omega)^H on the library's own output."""
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kds = [W.kpoint(cfg, 0)]
    for h, g, K2 in _gpu_real_axis(cfg, kds, OMEGA, ETA):
        chi = np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(len(OMEGA))])
    chi_o, _, _, _ = oracle_run(cfg, kds, True, omega=OMEGA, eta=ETA)
    for i in range(len(OMEGA)):
        assert rel_fro(chi[i], chi_o[i]) <= CHI_TOL, (i, rel_fro(chi[i], chi_o[i]))
    assert rel_fro(chi[3], chi[2].conj().T) <= 1e-13
    assert np.abs(chi[2] - chi[2].conj().T).max() > 1e-3 * np.abs(chi[2]).max()   # genuinely non-Hermitian


@pytest.mark.parametrize("batch", [16, 48])
def test_real_axis_ragged_batches_two_kpoints(batch):
    """Small batches (several launches, ragged last one), two k-points with different weights, no PAW."""
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kds = [W.kpoint(cfg, 0, occ=[0, 2, 3], unocc=range(0, 28, 2)), W.kpoint(cfg, 1, occ=[1], unocc=range(3, 26))]
    om = np.array([0.3, 1.7])
    for h, g, K2 in _gpu_real_axis(cfg, kds, om, 0.02, use_paw=False, batch=batch):
        chi = np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(2)])
    chi_o, _, _, _ = oracle_run(cfg, kds, False, omega=om, eta=0.02)
    for i in range(2):
        assert rel_fro(chi[i], chi_o[i]) <= CHI_TOL


def test_real_axis_at_z_equal_i_u_is_the_imaginary_axis_handle():
    """omega = 0, eta = u is the point i u: the real-axis handle must agree with the imaginary-axis one (two
    different weight kernels and read-outs, same accumulation)."""
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kds = [W.kpoint(cfg, 0)]
    om, _ = W.omega_grid(cfg.n_omega)
    chi_im, _, _, _ = gpu_run(cfg, kds, True, 0, want_ec=False)
    for i in (0, cfg.n_omega - 1):
        for h, g, K2 in _gpu_real_axis(cfg, kds, [0.0], float(om[i])):
            c = B.rpa_chi0_get(h, 0).cpu().numpy()
        assert rel_fro(c, chi_im[i]) <= 1e-13


def test_real_axis_errors():
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    for bad_eta in (0.0, -0.1, float("nan")):
        with pytest.raises(B.RpaError) as ei:
            B.rpa_chi0_create_real_axis(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), [0.1], bad_eta)
        assert ei.value.code == B.RPA_ERR_INVALID_ARG
    with pytest.raises(B.RpaError) as ei:
        B.rpa_chi0_create_real_axis(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), [0.1, float("inf")], 0.1)
    assert ei.value.code == B.RPA_ERR_INVALID_ARG
    h = B.rpa_chi0_create_real_axis(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), [0.1, 0.2], 0.1)
    try:
        g, K2 = B.rpa_chi0_gvectors(h)
        with pytest.raises(B.RpaError) as ei:
            B.rpa_ec_q(h, W.coulomb(K2))
        assert ei.value.code == B.RPA_ERR_UNSUPPORTED
        with pytest.raises(B.RpaError) as ei:   # two frequencies, four accumulator slots: index 2 is out of range
            B.rpa_chi0_get(h, 2)
        assert ei.value.code == B.RPA_ERR_INVALID_ARG
    finally:
        h.close()


def test_config1_real_axis_full_size_sampled():
    """BASELINE.json configs[1] at full grid / nG / projectors with 4 x 600 bands, 8 real frequencies (16 slots: the
    launch shape of the bench step), device-resident arrays; the oracle evaluates a sampled sub-list of the sphere."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[1]
    kds = [W.kpoint(cfg, 0, occ=[0, 5, 10, 11])]
    om = np.array([0.0, 0.05, 0.2, 0.35, 0.6, 1.0, 3.0, -0.35])
    for h, g, K2 in _gpu_real_axis(cfg, kds, om, 0.01, device_resident=True):
        ng = len(g)
        rng = np.random.default_rng(11)
        sel = set([0, 1, ng - 1, ng - 2, 63, 64, 65, 127, 128, (ng // 64) * 64 - 1, (ng // 64) * 64])
        sel |= set(rng.choice(ng, 48 - len(sel), replace=False).tolist())
        sel = np.array(sorted(sel))
        seld = torch.from_numpy(sel).to("cuda:0")
        chi_sel = {i: B.rpa_chi0_get(h, i)[seld][:, seld].cpu().numpy() for i in (1, 3, 7)}
        gsel = g[sel]
    chi_o, _, _, _ = oracle_run(cfg, kds, True, g=gsel, omega=om[[1, 3, 7]], eta=0.01)
    for j, i in enumerate((1, 3, 7)):
        assert rel_fro(chi_sel[i], chi_o[j]) <= CHI_TOL, (i, rel_fro(chi_sel[i], chi_o[j]))
    assert rel_fro(chi_sel[7], chi_sel[3].conj().T) <= 1e-12


def test_real_axis_streamed_kpoint_is_bitwise_the_single_call():
    """rpa_chi0_add_kpoint_begin / _pairs / _end on a real-axis handle (two accumulator slots per frequency): the same
    kernels in the same order as one rpa_chi0_add_kpoint call, so every slot agrees bit for bit."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    om = np.array([0.0, 0.4, -1.3])
    for h, g, K2 in _gpu_real_axis(cfg, [], om, ETA):
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
        dv = {k: torch.from_numpy(getattr(kd, k)).to("cuda:0") for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
        args = (kd.kweight, dv["psi_occ"], dv["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc, cfg.n_proj,
                dv["P_occ"], dv["P_unocc"], Qd, W.atom_positions(cfg))
        B.rpa_chi0_add_kpoint(h, *args)
        ref = [B.rpa_chi0_get(h, i).clone() for i in range(len(om))]
        B.rpa_chi0_reset(h)
        B.rpa_chi0_add_kpoint_begin(h, *args)
        n_u = dv["psi_unocc"].shape[0]
        for a, b in ((0, 7), (7, 8), (8, n_u)):
            B.rpa_chi0_add_kpoint_pairs(h, a, b)
        B.rpa_chi0_add_kpoint_end(h)
        for i in range(len(om)):
            assert torch.equal(B.rpa_chi0_get(h, i), ref[i]), i
        assert float(ref[1].abs().max()) > 0.0
