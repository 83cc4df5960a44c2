"""Parity of rpa_pw_to_grid (Eq. 10) and rpa_symmetry_remap (Eq. 11) against the CPU oracle,
through the C ABI.  Tolerance: 1e-12 relative to max |u| for the transform (sums of up to ~1e4
terms of unit-modulus phases in fp64: DESIGN.md section 5), bit-exact for the remap (pure data movement)."""
import numpy as np
import pytest

import oracle
from paper_1307_8052_b200 import workload as W
from tests.parity_util import gpu_run, rel_fro

pytestmark = pytest.mark.gpu


def _handle(cfg):
    from paper_1307_8052_b200 import binding as B
    om, wt = W.omega_grid(cfg.n_omega)
    return B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, int(cfg.n_proj.sum()), "cuda:0")


def _coeffs(cfg, k, bands):
    g = None
    C = []
    for b in bands:
        g, c = W.orbital_coefficients(cfg, k, b)
        C.append(c)
    return g, np.stack(C)


def test_pw_to_grid_toy_full_and_ragged_lists():
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    g, C = _coeffs(cfg, 0, range(5))
    h = _handle(cfg)
    try:
        u = B.rpa_pw_to_grid(h, g, torch.from_numpy(C).cuda()).cpu().numpy()
        want = oracle.pw_to_grid(cfg.grid, g, C).reshape(u.shape)
        assert np.abs(u - want).max() <= 1e-12 * np.abs(want).max()
        # an odd sub-list of plane waves in shuffled order, one band; a single plane wave; no plane wave at all
        sel = np.random.default_rng(1).permutation(len(g))[:37]
        u1 = B.rpa_pw_to_grid(h, g[sel], torch.from_numpy(C[:1, sel].copy()).cuda()).cpu().numpy()
        assert np.abs(u1 - oracle.pw_to_grid(cfg.grid, g[sel], C[:1, sel]).reshape(u1.shape)).max() <= 1e-12
        u2 = B.rpa_pw_to_grid(h, [[1, -2, 3]], torch.ones((1, 1), dtype=torch.complex128, device="cuda")).cpu().numpy()
        assert np.abs(u2 - oracle.pw_to_grid(cfg.grid, [[1, -2, 3]], [1.0]).reshape(u2.shape)).max() <= 1e-14
        u3 = B.rpa_pw_to_grid(h, np.zeros((0, 3), dtype=np.int32), torch.zeros((2, 0), dtype=torch.complex128, device="cuda"))
        assert float(u3.abs().max()) == 0.0
        with pytest.raises(B.RpaError) as ei:   # duplicate plane wave
            B.rpa_pw_to_grid(h, [[0, 0, 1], [0, 0, 1]], torch.ones((1, 2), dtype=torch.complex128, device="cuda"))
        assert ei.value.code == B.RPA_ERR_INVALID_ARG
    finally:
        h.close()


@pytest.mark.parametrize("grid", [(12, 10, 14), (9, 15, 7), (8, 24, 40), (24, 36, 16), (5, 6, 1), (16, 48, 96)])
def test_pw_to_grid_mixed_grids_all_points(grid):
    """Every kernel variant: axes with a radix-12 / radix-8 split (table-driven persistent kernel, several items per
    CTA) and axes without one (direct sums), boxes that start at every residue of the radix, 7 bands."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cell = np.array([[6.0, 0.2, 0.0], [0.1, 5.0, 0.3], [0.0, -0.2, 7.0]])
    cfg = W.custom_config(300 + sum(grid), cell, grid, (0.25, 0.0, 0.0), n_occ=2, n_unocc=3, ng_target=4, n_omega=2,
                          n_atoms=1, n_proj_per_atom=1, orb_ecut_ha=2.0)
    rng = np.random.default_rng(sum(grid))
    half = [max((n - 1) // 2, 0) for n in grid]
    lo = [-rng.integers(0, hf + 1) for hf in half]           # asymmetric box: lower corner at a random residue
    hi = [rng.integers(0, hf + 1) for hf in half]
    allg = np.array([(a, b, c) for a in range(lo[0], hi[0] + 1) for b in range(lo[1], hi[1] + 1)
                     for c in range(lo[2], hi[2] + 1)], dtype=np.int32)
    g = allg[rng.permutation(len(allg))[:max(1, (2 * len(allg)) // 3)]]
    C = rng.standard_normal((7, len(g))) + 1j * rng.standard_normal((7, len(g)))
    h = _handle(cfg)
    try:
        u = B.rpa_pw_to_grid(h, g, torch.from_numpy(C).cuda()).cpu().numpy()
    finally:
        h.close()
    want = oracle.pw_to_grid(cfg.grid, g, C).reshape(u.shape)
    assert np.abs(u - want).max() <= 1e-12 * np.abs(want).max()


def test_pw_to_grid_config1_full_size_sampled_points():
    """56x60x64 grid, ~9.4e3 plane waves (|G|^2/2 <= 6 Ha), 3 bands: the oracle sums at 400 sampled grid points
    (first / last point, plane and row boundaries, random rest); the generator's own orbital must also come out."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[1]
    bands = [0, 11, 300]
    g, C = _coeffs(cfg, 0, bands)
    h = _handle(cfg)
    try:
        u = B.rpa_pw_to_grid(h, g, torch.from_numpy(C).cuda()).cpu().numpy().reshape(len(bands), -1)
    finally:
        h.close()
    N = cfg.n_grid
    rng = np.random.default_rng(2)
    pts = np.unique(np.concatenate([[0, 1, 63, 64, 3839, 3840, N - 1, N - 64], rng.choice(N, 392, replace=False)]))
    want = oracle.pw_to_grid(cfg.grid, g, C, pts)
    assert np.abs(u[:, pts] - want).max() <= 1e-12 * np.abs(want).max()
    assert abs(np.mean(np.abs(u[0]) ** 2) - 1.0) < 1e-12                      # Parseval with sum |C|^2 = 1
    assert np.abs(u[1] - W.orbital(cfg, 0, 11).reshape(-1)).max() <= 1e-11   # numpy's inverse FFT route


def test_chi0_from_plane_wave_coefficients_matches_grid_route():
    """Config 0 end to end: orbitals made on the device from their coefficients give the same chi0 as the orbitals
    the generator makes on the host (both routes agree to rounding, so chi0 agrees to ~1e-13)."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    chi_ref, _, _, _ = gpu_run(cfg, [kd], False, 0, want_ec=False)
    g, Co = _coeffs(cfg, 0, range(cfg.n_occ))
    _, Cu = _coeffs(cfg, 0, range(cfg.n_occ, cfg.n_occ + cfg.n_unocc))
    h = _handle(cfg)
    try:
        po = B.rpa_pw_to_grid(h, g, torch.from_numpy(Co).cuda())
        pu = B.rpa_pw_to_grid(h, g, torch.from_numpy(Cu).cuda())
        B.rpa_chi0_add_kpoint(h, kd.kweight, po, pu, kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc)
        for i in range(cfg.n_omega):
            assert rel_fro(B.rpa_chi0_get(h, i).cpu().numpy(), chi_ref[i]) <= 1e-11
    finally:
        h.close()


def test_add_kpoint_host_pw_pipeline_against_the_oracle():
    """binding.add_kpoint_host_pw (upload coefficients, expand on the device, add) with PAW on, twice on one handle
    (buffers reused), against the oracle run on the generator's grid orbitals, and E_c(q)."""
    import torch
    from paper_1307_8052_b200 import binding as B
    from tests.parity_util import oracle_run
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    g_pw, Co, Cu = W.kpoint_coefficients(cfg, 0)
    om, wt = W.omega_grid(cfg.n_omega)
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, int(cfg.n_proj.sum()), "cuda:0")
    try:
        g, K2 = B.rpa_chi0_gvectors(h)
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
        pin = lambda a: torch.from_numpy(a).pin_memory()
        Cop, Cup, Pop, Pup = pin(Co), pin(Cu), pin(kd.P_occ), pin(kd.P_unocc)
        for _ in range(2):
            B.rpa_chi0_reset(h)
            nb = B.add_kpoint_host_pw(h, kd.kweight, g_pw, Cop, Cup, kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc,
                                      cfg.n_proj, Pop, Pup, Qd, W.atom_positions(cfg))
            assert nb == 16 * (Co.size + Cu.size + kd.P_occ.size + kd.P_unocc.size)
            chi = np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(cfg.n_omega)])
            ec, _ = B.rpa_ec_q(h, W.coulomb(K2))
    finally:
        h.close()
    chi_o, ec_o, _, _ = oracle_run(cfg, [kd], True)
    for i in range(cfg.n_omega):
        assert rel_fro(chi[i], chi_o[i]) <= 1e-10
    assert abs(ec - ec_o[0]) <= 1e-9 * abs(ec_o[0])


def test_pw_to_grid_index_table_is_kept_and_invalidated():
    """rpa_pw_to_grid keeps the index table of the last g_pw on the device: the same list again (after an add_kpoint has
    overwritten the handle's scratch), the same vectors in another order, another list and back must all give the
    oracle's orbitals."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    g, C = _coeffs(cfg, 0, range(3))
    perm = np.random.default_rng(5).permutation(len(g))
    sub = perm[:41]
    h = _handle(cfg)
    try:
        def check(gl, Cl):
            u = B.rpa_pw_to_grid(h, gl, torch.from_numpy(np.ascontiguousarray(Cl)).cuda()).cpu().numpy()
            want = oracle.pw_to_grid(cfg.grid, gl, Cl).reshape(u.shape)
            assert np.abs(u - want).max() <= 1e-12 * np.abs(want).max()
        check(g, C)
        check(g, C[::-1])                       # same list: the kept table
        B.add_kpoint_host(h, kd)                # pair densities run through the scratch the table used to live in
        check(g, C)
        check(g[perm], C[:, perm])              # same vectors, other order: another table
        check(g[sub], C[:, sub])                # a smaller box
        check(g, C)
        with pytest.raises(B.RpaError):         # a failed build leaves no table behind
            B.rpa_pw_to_grid(h, [[0, 0, 1], [0, 0, 1]], torch.ones((1, 2), dtype=torch.complex128, device="cuda"))
        check(g[sub], C[:, sub])
    finally:
        h.close()


def test_streamed_add_kpoint_is_bitwise_the_single_call():
    """rpa_chi0_add_kpoint_begin / _pairs / _end with ragged slices against ONE rpa_chi0_add_kpoint call on the same device
    orbitals: the same pair densities meet in the same rank-K update, so chi0 agrees bit for bit (PAW on).  Then the
    protocol errors: slices out of order, end before the last band, a second begin, add_kpoint while open, and a band
    set that is more than one batch."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    h = _handle(cfg)
    try:
        _, K2 = B.rpa_chi0_gvectors(h)
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).cuda()
        R = W.atom_positions(cfg)
        po, pu = torch.from_numpy(kd.psi_occ).cuda(), torch.from_numpy(kd.psi_unocc).cuda()
        Po, Pu = torch.from_numpy(kd.P_occ).cuda(), torch.from_numpy(kd.P_unocc).cuda()
        args = (kd.kweight, po, pu, kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc, cfg.n_proj, Po, Pu, Qd, R)
        B.rpa_chi0_add_kpoint(h, *args)
        ref = [B.rpa_chi0_get(h, i).clone() for i in range(cfg.n_omega)]
        n_u = pu.shape[0]
        for cuts in ([0, n_u], [0, 1, 2, 9, n_u], [0, 5, 5, 20, n_u]):
            B.rpa_chi0_reset(h)
            B.rpa_chi0_add_kpoint_begin(h, *args)
            for a, b in zip(cuts[:-1], cuts[1:]):
                B.rpa_chi0_add_kpoint_pairs(h, a, b)
                B.rpa_chi0_get(h, 0)   # other calls are allowed while the k-point is open
            B.rpa_chi0_add_kpoint_end(h)
            for i in range(cfg.n_omega):
                assert torch.equal(B.rpa_chi0_get(h, i), ref[i]), (cuts, i)
        # protocol errors
        for call in (lambda: B.rpa_chi0_add_kpoint_pairs(h, 0, 1), lambda: B.rpa_chi0_add_kpoint_end(h)):
            with pytest.raises(B.RpaError) as ei:   # nothing open
                call()
            assert ei.value.code == B.RPA_ERR_INVALID_ARG
        B.rpa_chi0_reset(h)
        B.rpa_chi0_add_kpoint_begin(h, *args)
        for call in (lambda: B.rpa_chi0_add_kpoint_begin(h, *args), lambda: B.rpa_chi0_add_kpoint(h, *args),
                     lambda: B.rpa_chi0_add_kpoint_pairs(h, 1, 2), lambda: B.rpa_chi0_add_kpoint_pairs(h, 0, n_u + 1)):
            with pytest.raises(B.RpaError) as ei:
                call()
            assert ei.value.code == B.RPA_ERR_INVALID_ARG
        B.rpa_chi0_add_kpoint_pairs(h, 0, 3)
        with pytest.raises(B.RpaError) as ei:       # ended early: nothing is added, the k-point is closed
            B.rpa_chi0_add_kpoint_end(h)
        assert ei.value.code == B.RPA_ERR_INVALID_ARG
        assert float(B.rpa_chi0_get(h, 0).abs().max()) == 0.0
        B.rpa_chi0_add_kpoint(h, *args)
        assert torch.equal(B.rpa_chi0_get(h, 1), ref[1])
    finally:
        h.close()
    # more than one batch: 4 x 28 transitions on a handle created for 64 per batch
    om, wt = W.omega_grid(cfg.n_omega)
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 64, int(cfg.n_proj.sum()), "cuda:0")
    try:
        with pytest.raises(B.RpaError) as ei:
            B.rpa_chi0_add_kpoint_begin(h, *args)
        assert ei.value.code == B.RPA_ERR_UNSUPPORTED
        B.rpa_chi0_add_kpoint(h, *args)             # nothing was left open
    finally:
        h.close()


def test_add_kpoint_host_pw_in_two_calls_agrees_with_one():
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    g_pw, Co, Cu = W.kpoint_coefficients(cfg, 0)
    h = _handle(cfg)
    try:
        _, K2 = B.rpa_chi0_gvectors(h)
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
        pin = lambda a: torch.from_numpy(a).pin_memory()
        Cop, Cup, Pop, Pup = pin(Co), pin(Cu), pin(kd.P_occ), pin(kd.P_unocc)
        res = []
        for n_calls, n_slices in ((1, 4), (2, 4), (3, 7), (1, 1)):
            B.rpa_chi0_reset(h)
            B.add_kpoint_host_pw(h, kd.kweight, g_pw, Cop, Cup, kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc, cfg.n_proj, Pop,
                                 Pup, Qd, W.atom_positions(cfg), n_slices=n_slices, n_calls=n_calls)
            res.append(np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(cfg.n_omega)]))
    finally:
        h.close()
    for r in res[1:]:
        for i in range(cfg.n_omega):
            assert rel_fro(r[i], res[0][i]) <= 1e-13


@pytest.mark.parametrize("M,tr", [(np.eye(3, dtype=int), True), (-np.eye(3, dtype=int), False),
                                  ([[0, -1, 0], [1, 0, 0], [0, 0, 1]], False), ([[0, 1, 0], [1, 0, 0], [0, 0, -1]], True)])
def test_symmetry_remap_bit_exact(M, tr):
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]   # cubic 16^3 grid: every point-group operation maps it onto itself
    kd = W.kpoint(cfg, 0, occ=[0, 1], unocc=[0])
    h = _handle(cfg)
    try:
        out = B.rpa_symmetry_remap(h, torch.from_numpy(kd.psi_occ).cuda(), M, tr).cpu().numpy()
    finally:
        h.close()
    assert np.array_equal(out, oracle.symmetry_remap(cfg.grid, M, tr, kd.psi_occ))


def test_symmetry_remap_rejects_incompatible_operation():
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[1]   # 56 x 60 x 64: swapping x and z does not map the grid onto itself
    h = _handle(cfg)
    try:
        psi = torch.zeros((1,) + tuple(cfg.grid), dtype=torch.complex128, device="cuda")
        with pytest.raises(B.RpaError) as ei:
            B.rpa_symmetry_remap(h, psi, [[0, 0, 1], [0, 1, 0], [1, 0, 0]])
        assert ei.value.code == B.RPA_ERR_UNSUPPORTED
        out = B.rpa_symmetry_remap(h, psi, [[-1, 0, 0], [0, 1, 0], [0, 0, -1]])   # a mirror pair is fine
        assert out.shape == psi.shape
    finally:
        h.close()
