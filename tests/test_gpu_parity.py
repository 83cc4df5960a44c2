"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances are BASELINE.json north_star's: chi0 relative Frobenius error <= 1e-10 per frequency, E_c(q)
relative error <= 1e-9.  All tests need a B200 (``-m gpu``)."""
import numpy as np
import pytest

from paper_1307_8052_b200 import workload as W
from tests.parity_util import gpu_run, oracle_run, rel_fro

pytestmark = pytest.mark.gpu

CHI_TOL = 1e-10
EC_TOL = 1e-9


def _compare(cfg, kds, use_paw=True, max_batch_pairs=0):
    chi_g, ec_g, g_g, K2_g = gpu_run(cfg, kds, use_paw, max_batch_pairs)
    chi_o, ec_o, g_o, K2_o = oracle_run(cfg, kds, use_paw)
    assert g_g.shape == g_o.shape and (g_g == g_o).all(), "sphere / ordering differs"
    assert np.allclose(K2_g, K2_o, rtol=1e-13)
    for i in range(cfg.n_omega):
        err = rel_fro(chi_g[i], chi_o[i])
        assert err <= CHI_TOL, f"omega {i}: rel Frobenius error {err:.3e}"
        # and element by element: no element (far off-diagonal ones included) further from the oracle than 1e-10 of the
        # largest element -- a norm dominated by the diagonal cannot hide a wrong small element behind it
        worst = float(np.abs(chi_g[i] - chi_o[i]).max() / np.abs(chi_o[i]).max())
        assert worst <= CHI_TOL, f"omega {i}: largest element error {worst:.3e} of the largest element"
    assert abs(ec_g[0] - ec_o[0]) <= EC_TOL * abs(ec_o[0]), (ec_g[0], ec_o[0])
    # e(omega) = ln det + Tr is a cancelling difference at large omega: compare on the scale of the largest term
    assert np.allclose(ec_g[1], ec_o[1], rtol=EC_TOL, atol=1e-12 * np.abs(ec_o[1]).max())
    return chi_g


def test_tiny_skewed_cell_ragged(tiny_cfg):
    """6x4x8 grid, skewed cell, 2x5 bands, 3 frequencies, 2 atoms x 3 projectors: every tail is ragged."""
    _compare(tiny_cfg, [W.kpoint(tiny_cfg, 0)])


@pytest.mark.parametrize("ng_target", [63, 64, 65, 127, 129, 191, 193, 257])
def test_sphere_sizes_around_the_tile_edges(ng_target):
    """nG on and next to multiples of the rank-K tile (64) and of its 8-row warp blocks: one or two rows / columns in the
    last tile, a full last tile, a diagonal tile that is the ragged one -- every element of chi0 and E_c(q) against the
    oracle (skewed cell, 20^3 grid, 3 x 11 bands in batches of 32 so that several ragged batches add up, PAW on)."""
    cell = np.array([[7.0, 0.3, 0.0], [0.2, 7.5, 0.1], [0.0, -0.4, 8.0]])
    cfg = W.custom_config(300 + ng_target, cell, (20, 20, 20), (0.25, 0.1, 0.0), n_occ=3, n_unocc=11, ng_target=ng_target,
                          n_omega=3, n_atoms=2, n_proj_per_atom=2, orb_ecut_ha=3.0)
    chi = _compare(cfg, [W.kpoint(cfg, 0)], max_batch_pairs=32)
    assert chi.shape[1] == ng_target


def test_config0_toy_full():
    cfg = W.CONFIGS[0]
    chi = _compare(cfg, [W.kpoint(cfg, 0)])
    for i in range(cfg.n_omega):  # Hermitian by construction, negative semidefinite on the imaginary axis
        assert np.array_equal(chi[i], chi[i].conj().T)
        assert np.linalg.eigvalsh(chi[i]).max() <= 1e-13 * np.abs(chi[i]).max()


def test_config0_no_paw():
    cfg = W.CONFIGS[0]
    _compare(cfg, [W.kpoint(cfg, 0)], use_paw=False)


@pytest.mark.parametrize("batch", [16, 48, 100])
def test_batch_size_invariance(batch):
    """Results must not depend on the internal grouping of transitions (the paper's Nu)."""
    cfg = W.CONFIGS[0]
    kds = [W.kpoint(cfg, 0)]
    a, _, _, _ = gpu_run(cfg, kds, True, 0, want_ec=False)
    b, _, _, _ = gpu_run(cfg, kds, True, batch, want_ec=False)
    for i in range(cfg.n_omega):
        assert rel_fro(b[i], a[i]) <= 1e-12


def test_additivity_over_calls():
    """Splitting bands over several add_kpoint calls gives the same chi0."""
    cfg = W.CONFIGS[0]
    full = [W.kpoint(cfg, 0)]
    parts = [W.kpoint(cfg, 0, occ=[0, 1], unocc=range(0, 11)), W.kpoint(cfg, 0, occ=[0, 1], unocc=range(11, 28)),
             W.kpoint(cfg, 0, occ=[2, 3])]
    a, _, _, _ = gpu_run(cfg, full, True, 0, want_ec=False)
    b, _, _, _ = gpu_run(cfg, parts, True, 0, want_ec=False)
    for i in range(cfg.n_omega):
        assert rel_fro(b[i], a[i]) <= 1e-12


@pytest.mark.parametrize("grid,q", [((12, 10, 14), (0.25, 0.0, 0.5)), ((9, 15, 7), (0.1, 0.2, -0.3)),
                                    ((8, 1, 6), (0.5, 0.0, 0.0)), ((5, 6, 1), (0.0, 0.25, 0.0))])
def test_mixed_radix_grids(grid, q):
    """Grid lengths with factors 2, 3, 5, 7 and degenerate axes of length 1."""
    cell = np.array([[6.0, 0.2, 0.0], [0.1, 5.0, 0.3], [0.0, -0.2, 7.0]])
    cfg = W.custom_config(200 + sum(grid), cell, grid, q, n_occ=3, n_unocc=7, ng_target=12, n_omega=4, n_atoms=2,
                          n_proj_per_atom=2, orb_ecut_ha=2.0)
    _compare(cfg, [W.kpoint(cfg, 0)])


def test_config2_bulk_two_kpoints_slice():
    """24^3 fcc grid, nG = 401 (ragged 64-tile tail), 16 frequencies, 3 atoms x 8 projectors; 2 k-points,
    3 occupied x 45 unoccupied bands each."""
    cfg = W.CONFIGS[2]
    kds = [W.kpoint(cfg, k, occ=[0, 3, 7], unocc=range(0, 300, 7)[:45]) for k in (0, 1)]
    _compare(cfg, kds)


def test_config1_molecule_slice():
    """56x60x64 grid (radices 7, 5, 3), nG = 1200, 2 occupied x 37 unoccupied bands."""
    cfg = W.CONFIGS[1]
    kds = [W.kpoint(cfg, 0, occ=[0, 11], unocc=range(0, 600, 16)[:37])]
    _compare(cfg, kds)


def _big_config_slice(cfg, occ, unocc, n_sample, omegas=(0, 7, 15), k_list=(0, 1), device_resident=False, modes=(None,),
                      max_batch=0, want_batches=None):
    """Configs 3 / 4 at full grid, nG, omega count and atoms, on a band slice (a full oracle run costs hours to a
    day of CPU).  The oracle evaluates chi0 on a sampled sub-list of the sphere (every element of
    Eq. 17 is an independent sum, so chi0 restricted to those G is exactly the chi0 of those G); the sample holds
    the first / last G and both sides of several 64-tile boundaries.  E_c(q), which needs the whole matrix, is
    checked against the eigenvalue route sum_i ln(1 - l_i) + l_i on the library's own chi0 (numpy eigvalsh).
    modes: one GPU run per entry (None = the library's default rank-K kernel, else (mode, digits) for
    rpa_chi0_set_rank_k_mode), every one compared with the SAME oracle result; the E_c check runs for the first.
    want_batches: per mode, the (FP64, int8) batch counts rpa_chi0_rank_k_batches must report."""
    import torch
    from paper_1307_8052_b200 import binding as B
    om, wt = W.omega_grid(cfg.n_omega)
    ptot = int(cfg.n_proj.sum())
    kds = [W.kpoint(cfg, k, occ=occ, unocc=unocc) for k in k_list]
    results = []
    sel = g = None
    for im, mode in enumerate(modes):
        h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, max_batch, ptot, "cuda:0")
        try:
            if mode is not None:
                B.rpa_chi0_set_rank_k_mode(h, *mode)
            g, K2 = B.rpa_chi0_gvectors(h)
            ng = len(g)
            rng = np.random.default_rng(7)
            sel = set([0, 1, ng - 1, ng - 2, 63, 64, 65, 127, 128, (ng // 64) * 64 - 1, (ng // 64) * 64])
            sel |= set(rng.choice(ng, n_sample - len(sel), replace=False).tolist())
            sel = np.array(sorted(s for s in sel if 0 <= s < ng))
            Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
            R = W.atom_positions(cfg)
            for kd in kds:
                if device_resident:  # exactly what bench.py's timed step does: arrays already in HBM, one call per k-point
                    dv = {k: torch.from_numpy(getattr(kd, k)).to("cuda:0") for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
                    B.rpa_chi0_add_kpoint(h, kd.kweight, dv["psi_occ"], dv["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ,
                                          kd.f_unocc, cfg.n_proj, dv["P_occ"], dv["P_unocc"], Qd, R)
                    B.rpa_chi0_sync(h)
                    del dv
                else:
                    B.add_kpoint_host(h, kd, cfg.n_proj, Qd, R)
            if want_batches is not None:
                assert B.rpa_chi0_rank_k_batches(h) == want_batches[im], (mode, B.rpa_chi0_rank_k_batches(h))
            seld = torch.from_numpy(sel).to("cuda:0")
            chi_sel, chi_full = {}, {}
            for i in omegas:
                c = B.rpa_chi0_get(h, i)
                chi_sel[i] = c[seld][:, seld].cpu().numpy()
                if im == 0 and i in (omegas[0], omegas[-1]):
                    chi_full[i] = c.cpu().numpy()
                del c
            v = W.coulomb(K2)
            ec, e = B.rpa_ec_q(h, v)
            results.append((chi_sel, chi_full, ec, e, v))
        finally:
            h.close()
        torch.cuda.empty_cache()
    chi_o, _, g_o, _ = oracle_run(cfg, kds, True, want_ec=False, g=g[sel])
    for (chi_sel, _, _, _, _), mode in zip(results, modes):
        for i in omegas:
            err = rel_fro(chi_sel[i], chi_o[i])
            assert err <= CHI_TOL, f"mode {mode}, omega {i}: rel Frobenius error on the sampled G {err:.3e}"
            # and element by element on the sample: every sampled element within 1e-9 of the sample's largest
            # (a wrong far off-diagonal element cannot hide behind the diagonal's norm)
            assert np.abs(chi_sel[i] - chi_o[i]).max() <= 1e-9 * np.abs(chi_o[i]).max(), (mode, i)
    _, chi_full, ec, e, v = results[0]
    d = np.sqrt(v)
    for i, c in chi_full.items():
        assert np.array_equal(c, c.conj().T)
        lam = np.linalg.eigvalsh(d[:, None] * c * d[None, :])
        assert lam.max() <= 1e-12 * np.abs(lam).max()          # negative semidefinite
        want = float(np.sum(np.log1p(-lam) + lam))
        assert abs(e[i] - want) <= 1e-9 * max(abs(want), np.abs(e).max() * 1e-3), (i, e[i], want)
    assert np.isfinite(ec) and ec < 0.0
    for r in results[1:]:   # E_c(q) of the other modes against the first
        assert abs(r[2] - ec) <= 1e-10 * abs(ec)


def test_config3_slab_slice():
    """40x40x168 grid (radices 8,7,3 / 8,5), nG = 3004, 16 omega, 10 atoms x 18 projectors, metallic smearing;
    2 k-points x 3 occupied (lowest, middle, highest) x 23 unoccupied (strided, includes the band nearest mu)."""
    cfg = W.CONFIGS[3]
    _big_config_slice(cfg, occ=[0, 31, 63], unocc=list(range(0, 1500, 68))[:23], n_sample=160)


def test_config4_large_slab_slice():
    """48x48x192 grid, nG = 5001 (chi0 6.4 GB resident), 18 atoms x 18 projectors; 2 k-points x 2 occupied x 13
    unoccupied."""
    cfg = W.CONFIGS[4]
    _big_config_slice(cfg, occ=[0, 119], unocc=list(range(0, 3000, 240))[:13], n_sample=120)


def _all_rank_k_modes():
    from paper_1307_8052_b200 import binding as B
    return (None, (B.RPA_RANK_K_FP64_4M, 0), (B.RPA_RANK_K_I8, 7), (B.RPA_RANK_K_I8, 8))


def test_config3_large_batch_every_rank_k_mode():
    """What a real configs[3] run launches: one batch of >= 1024 transitions (1 occupied x 1031 unoccupied, odd count,
    Kpad = 1056) at full grid / nG = 3004 / 16 omega / 10 x 18 projectors, device-resident, for every rank-K mode against
    ONE oracle run on 120 sampled G.  FP64 3M (default): 1128 tiles x 16 omega in whole waves plus a K-sliced tail launch;
    int8 (picked by the library's own thresholds, no ALL_BATCHES flag): 24 row blocks per half, odd tile rows with padding
    tiles, and -- with max_batch_pairs = 1056 sizing the scratch -- the frequencies in three groups (6, 6, 4), as at the
    default batch of 8192 (Eq. 17 / Eq. 20)."""
    cfg = W.CONFIGS[3]
    _big_config_slice(cfg, occ=[31], unocc=list(range(3, 1034)), n_sample=120, k_list=(0,),
                      device_resident=True, modes=_all_rank_k_modes(), max_batch=1056,
                      want_batches=((1, 0), (1, 0), (0, 1), (0, 1)))


def test_config4_large_batch_every_rank_k_mode():
    """The same for configs[4]: 48x48x192 grid, nG = 5001 (79 column blocks, 40 row blocks per half), 18 x 18 projectors,
    1 occupied x 1031 unoccupied bands in one batch."""
    cfg = W.CONFIGS[4]
    _big_config_slice(cfg, occ=[59], unocc=list(range(0, 3000, 2))[:1031], n_sample=100, k_list=(0,),
                      device_resident=True, modes=_all_rank_k_modes(), max_batch=1056,
                      want_batches=((1, 0), (1, 0), (0, 1), (0, 1)))


def test_config1_full_size_bench_configuration():
    """BASELINE.json configs[1] at FULL size (56x60x64, 12 x 600 bands = 7200 transitions, nG = 1200, 16 omega,
    2 atoms x 13 projectors) in the launch configuration bench.py times (device-resident arrays, default
    max_batch_pairs, one add_kpoint call).  The oracle evaluates chi0 on a sampled sub-list of the sphere for three
    frequencies (every element of Eq. 17 is an independent sum); E_c(q) is checked by the eigenvalue route."""
    cfg = W.CONFIGS[1]
    _big_config_slice(cfg, occ=None, unocc=None, n_sample=72, k_list=(0,), device_resident=True)


def test_pipelined_host_upload_matches_single_call():
    """binding.add_kpoint_host with pinned inputs uploads the unoccupied bands in slices on a side stream and adds
    every slice with its own call; the result must equal the one-call result (additivity) to rounding."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    a, _, _, _ = gpu_run(cfg, [kd], True, 0, want_ec=False)
    om, wt = W.omega_grid(cfg.n_omega)
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, int(cfg.n_proj.sum()), "cuda:0")
    try:
        g, K2 = B.rpa_chi0_gvectors(h)
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
        pinned = {k: torch.from_numpy(getattr(kd, k)).pin_memory() for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
        for _ in range(2):   # twice: the alternating buffers and their events are reused
            B.rpa_chi0_reset(h)
            nb = B.add_kpoint_host(h, kd, cfg.n_proj, Qd, W.atom_positions(cfg), pinned=pinned, chunk_bands=5)
            assert nb == sum(t.numel() * 16 for t in pinned.values())
            for i in range(cfg.n_omega):
                b = B.rpa_chi0_get(h, i).cpu().numpy()
                assert rel_fro(b, a[i]) <= 1e-12
    finally:
        h.close()


def test_four_multiplication_rank_k_path_still_agrees(tiny_cfg):
    """rpa_chi0_set_rank_k_mode(RPA_RANK_K_FP64_4M) selects rank_k_kernel<true>, the 4-multiplication real-view kernel
    that rank_k3m_kernel replaced for the chi0 accumulation; it stays the reference form of the update (and its <false>
    variant serves the Cholesky), so its parity with the oracle is kept under test."""
    from paper_1307_8052_b200 import binding as B
    cfg2 = W.CONFIGS[2]
    cases = [(W.CONFIGS[0], [W.kpoint(W.CONFIGS[0], 0)]), (tiny_cfg, [W.kpoint(tiny_cfg, 0)]),
             (cfg2, [W.kpoint(cfg2, k, occ=[0, 3, 7], unocc=range(0, 300, 7)[:45]) for k in (0, 1)])]
    for cfg, kds in cases:
        chi_g, ec_g, _, _ = gpu_run(cfg, kds, True, rank_k_mode=(B.RPA_RANK_K_FP64_4M, 0))
        chi_o, ec_o, _, _ = oracle_run(cfg, kds, True)
        for i in range(cfg.n_omega):
            assert rel_fro(chi_g[i], chi_o[i]) <= CHI_TOL
        assert abs(ec_g[0] - ec_o[0]) <= EC_TOL * abs(ec_o[0])


def test_rank_k_mode_setter_validates():
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    om, wt = W.omega_grid(cfg.n_omega)
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, 0, "cuda:0")
    try:
        for mode, digits in ((7, 0), (B.RPA_RANK_K_I8, 5), (B.RPA_RANK_K_I8, 9), (B.RPA_RANK_K_I8 | 0x800, 7),
                             (B.RPA_RANK_K_FP64_3M | B.RPA_RANK_K_FLAG_ALL_BATCHES, 0)):
            with pytest.raises(B.RpaError) as ei:
                B.rpa_chi0_set_rank_k_mode(h, mode, digits)
            assert ei.value.code == B.RPA_ERR_INVALID_ARG
        for mode, digits in ((B.RPA_RANK_K_I8, 0), (B.RPA_RANK_K_I8 | B.RPA_RANK_K_FLAG_NO_CLUSTER, 8),
                             (B.RPA_RANK_K_FP64_4M, 0), (B.RPA_RANK_K_FP64_3M, 0)):
            B.rpa_chi0_set_rank_k_mode(h, mode, digits)
        assert B.rpa_chi0_rank_k_batches(h) == (0, 0)
    finally:
        h.close()


def test_config4_batch_spanning_two_pair_density_launches():
    """A default-size batch of configs[4] (8 x 1024 = 8192 transitions, 48x48x192 grid) needs 5 GB of pair-density scratch, more
    than the 4 GB the library gives it, so the batch is transformed by TWO launches of the z/y and x kernels, the second
    starting in the middle of an occupied row (pair 7050 = row 6, column 906).  The same k-point added with
    max_batch_pairs = 4096 (two batches of four whole rows, one launch each) must give the same chi0 to rounding; that
    configuration's kernels are compared with the oracle by test_config4_large_batch_every_rank_k_mode."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[4]
    om, wt = W.omega_grid(cfg.n_omega)
    ptot = int(cfg.n_proj.sum())
    occ, unocc = list(range(8)), list(range(1024))
    g_pw, C_o, C_u = W.kpoint_coefficients(cfg, 0, occ, unocc)
    eps, f = W.eigenvalues(cfg, 0)
    P = W.projections(cfg, 0)
    bo, bu = np.asarray(occ), np.asarray(unocc) + cfg.n_occ
    c = np.ascontiguousarray
    out = []
    for batch in (0, 4096):
        h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, batch, ptot, "cuda:0")
        try:
            g, K2 = B.rpa_chi0_gvectors(h)
            psi_o = B.rpa_pw_to_grid(h, g_pw, torch.from_numpy(C_o).to("cuda:0"))
            psi_u = B.rpa_pw_to_grid(h, g_pw, torch.from_numpy(C_u).to("cuda:0"))
            Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
            B.rpa_chi0_add_kpoint(h, 0.125, psi_o, psi_u, c(eps[bo]), c(eps[bu]), c(f[bo]), c(f[bu]), cfg.n_proj,
                                  torch.from_numpy(c(P[bo])).to("cuda:0"), torch.from_numpy(c(P[bu])).to("cuda:0"), Qd,
                                  W.atom_positions(cfg))
            assert B.rpa_chi0_rank_k_batches(h)[0] == (1 if batch == 0 else 2)
            chi = B.rpa_chi0_get(h, 5)
            sel = torch.arange(0, chi.shape[0], 7, device="cuda:0")
            out.append(chi[sel][:, sel].cpu().numpy())
            del chi, psi_o, psi_u, Qd
        finally:
            h.close()
        torch.cuda.empty_cache()
    assert rel_fro(out[0], out[1]) <= 1e-12
    assert np.abs(out[0] - out[1]).max() <= 1e-11 * np.abs(out[1]).max()


def _full_config_every_element(cfg, k_list):
    """A BASELINE config at FULL size -- every k-point in k_list with all its bands, default batching, device-resident
    arrays, one rpa_chi0_add_kpoint per k-point: the launch configuration bench.py times -- against a FULL oracle run:
    every element of every frequency (relative Frobenius <= 1e-10 and largest element error <= 1e-10 of the largest
    element) and E_c(q), e(omega) against the oracle's own unblocked Cholesky."""
    import torch
    from paper_1307_8052_b200 import binding as B
    import oracle
    om, wt = W.omega_grid(cfg.n_omega)
    ptot = int(cfg.n_proj.sum())
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, ptot, "cuda:0")
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    try:
        g, K2 = B.rpa_chi0_gvectors(h)
        assert (g == orc.g).all()
        Q = W.paw_Q(cfg, K2)
        Qd = torch.from_numpy(Q).to("cuda:0")
        R = W.atom_positions(cfg)
        for k in k_list:
            kd = W.kpoint(cfg, k)
            dv = {n: torch.from_numpy(getattr(kd, n)).to("cuda:0") for n in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
            B.rpa_chi0_add_kpoint(h, kd.kweight, dv["psi_occ"], dv["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc,
                                  cfg.n_proj, dv["P_occ"], dv["P_unocc"], Qd, R)
            orc.add_kpoint(kd, cfg.n_proj, Q, R)   # the CPU works while the GPU does
            B.rpa_chi0_sync(h)
            del dv
        assert B.rpa_chi0_rank_k_batches(h)[1] == 0   # the default FP64 kernel
        chi_o = orc.get()
        for i in range(cfg.n_omega):
            c = B.rpa_chi0_get(h, i).cpu().numpy()
            err = rel_fro(c, chi_o[i])
            assert err <= CHI_TOL, f"omega {i}: rel Frobenius error {err:.3e}"
            worst = float(np.abs(c - chi_o[i]).max() / np.abs(chi_o[i]).max())
            assert worst <= CHI_TOL, f"omega {i}: largest element error {worst:.3e}"
        v = W.coulomb(K2)
        ec, e = B.rpa_ec_q(h, v)
        ec_o, e_o = orc.ec_q(v)
        assert abs(ec - ec_o) <= EC_TOL * abs(ec_o), (ec, ec_o)
        assert np.allclose(e, e_o, rtol=EC_TOL, atol=1e-12 * np.abs(e_o).max())
    finally:
        h.close()


def test_config1_full_size_every_element():
    """configs[1] in full (7200 transitions, 56x60x64 grid, nG = 1200, 16 omega, PAW): all 16 x 1200 x 1200 elements and E_c(q)
    against a full oracle run (about half a minute of CPU)."""
    _full_config_every_element(W.CONFIGS[1], [0])


def test_config2_full_every_kpoint_every_element():
    """configs[2] in full: all 64 k-points x 8 x 300 bands = 153 600 transitions (24^3 grid, nG = 401, 16 omega, PAW): all
    elements and E_c(q) against a full oracle run (about a minute of CPU)."""
    cfg = W.CONFIGS[2]
    _full_config_every_element(cfg, list(range(cfg.n_k)))
