"""The int8-sliced rank-K update (csrc/rank_k_i8.cuh: tcgen05.mma.kind::i8 on error-free digit slices of the FP64
operands) against the CPU oracle, element by element, through the C ABI.  The library picks it by itself for large
batches (nG >= 768, K >= 1024: tests/test_gpu_parity.py::test_config1_full_size_bench_configuration runs it in the
bench configuration); here RPA_RANK_K_I8=1 forces it on small problems so that the oracle can check every element,
ragged tiles and several batches, and RPA_RANK_K_FP64=1 keeps the FP64 tensor kernel covered at full size.
The environment is read by rpa_chi0_create."""
import numpy as np
import pytest

from paper_1307_8052_b200 import workload as W
from tests.parity_util import gpu_run, oracle_run, rel_fro

pytestmark = pytest.mark.gpu

CHI_TOL, EC_TOL = 1e-10, 1e-9   # BASELINE.json north_star


@pytest.mark.parametrize("digits,bound", [(7, 2e-13), (6, 3e-11)])
def test_config0_all_elements(monkeypatch, digits, bound):
    """155 G vectors (two ragged 128-row blocks per half, three 64-column blocks), 4 x 28 transitions, PAW on.  The
    error bound of the scheme (2^-(6 + 7 (digits - 1)) of the row scale per operand) is checked as well
    as the path's tolerance."""
    monkeypatch.setenv("RPA_RANK_K_I8", "1")
    monkeypatch.setenv("RPA_RANK_K_I8_DIGITS", str(digits))
    cfg = W.CONFIGS[0]
    kds = [W.kpoint(cfg, 0)]
    chi, ec, _, _ = gpu_run(cfg, kds, True, 0, want_ec=True)
    chi_o, ec_o, _, _ = oracle_run(cfg, kds, True)
    for i in range(cfg.n_omega):
        err = rel_fro(chi[i], chi_o[i])
        assert err <= min(CHI_TOL, bound), (i, err)
        assert np.array_equal(chi[i], chi[i].conj().T)
    assert abs(ec[0] - ec_o[0]) <= EC_TOL * abs(ec_o[0])


@pytest.mark.parametrize("batch", [16, 48])
def test_small_batches_two_kpoints_no_paw(monkeypatch, batch):
    """K = 16 / 48 pairs per batch (one or two 32-pair K blocks per half, zero-padded rows), two k-points."""
    monkeypatch.setenv("RPA_RANK_K_I8", "1")
    cfg = W.CONFIGS[0]
    kds = [W.kpoint(cfg, 0, occ=[0, 2, 3], unocc=range(0, 28, 2)), W.kpoint(cfg, 1, occ=[1], unocc=range(3, 26))]
    chi, _, _, _ = gpu_run(cfg, kds, False, batch, want_ec=False)
    chi_o, _, _, _ = oracle_run(cfg, kds, False, want_ec=False)
    for i in range(cfg.n_omega):
        assert rel_fro(chi[i], chi_o[i]) <= 1e-12


def test_skewed_cell_mixed_grid_and_smearing(monkeypatch):
    """401 G vectors of config 2 (ragged last blocks), metallic-style weights of very different sizes in one row."""
    monkeypatch.setenv("RPA_RANK_K_I8", "1")
    cfg = W.CONFIGS[2]
    kds = [W.kpoint(cfg, 0, occ=[0, 3, 7], unocc=range(0, 300, 7))]
    chi, ec, _, _ = gpu_run(cfg, kds, True, 0, want_ec=True)
    chi_o, ec_o, _, _ = oracle_run(cfg, kds, True)
    for i in range(cfg.n_omega):
        assert rel_fro(chi[i], chi_o[i]) <= 1e-12
    assert abs(ec[0] - ec_o[0]) <= EC_TOL * abs(ec_o[0])


def test_int8_and_fp64_kernels_agree_at_full_size(monkeypatch):
    """configs[1], all 7200 transitions, device-resident: the default (int8 slices, 7 digits) against the FP64 tensor
    kernel (RPA_RANK_K_FP64=1) on the whole matrices; both are checked against the oracle elsewhere."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[1]
    kd = W.kpoint(cfg, 0)
    om, wt = W.omega_grid(cfg.n_omega)
    dv = {k: torch.from_numpy(getattr(kd, k)).to("cuda:0") for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
    out = {}
    for mode in ("i8", "fp64"):
        if mode == "fp64":
            monkeypatch.setenv("RPA_RANK_K_FP64", "1")
        h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, int(cfg.n_proj.sum()), "cuda:0")
        try:
            g, K2 = B.rpa_chi0_gvectors(h)
            Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
            B.rpa_chi0_set_profiling(h, True)
            B.rpa_chi0_add_kpoint(h, kd.kweight, dv["psi_occ"], dv["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc,
                                  cfg.n_proj, dv["P_occ"], dv["P_unocc"], Qd, W.atom_positions(cfg))
            B.rpa_chi0_sync(h)
            ms, n = B.rpa_chi0_stage_times(h)
            assert (n[5] > 0) == (mode == "i8")   # the kernel that ran is the one the mode names
            out[mode] = ([B.rpa_chi0_get(h, i).cpu().numpy() for i in (0, 7, 15)], B.rpa_ec_q(h, W.coulomb(K2))[0])
        finally:
            h.close()
    for a, b in zip(out["i8"][0], out["fp64"][0]):
        assert rel_fro(a, b) <= 2e-13
    assert abs(out["i8"][1] - out["fp64"][1]) <= 1e-13 * abs(out["fp64"][1])
