"""Edge cases and error behaviour of the C ABI on a real device (include/rpa_chi0.h: "errors" paragraph)."""
import numpy as np
import pytest

from paper_1307_8052_b200 import workload as W
from tests.parity_util import oracle_run, rel_fro

pytestmark = pytest.mark.gpu


def _handle(cfg, ptot=None, batch=0):
    from paper_1307_8052_b200 import binding as B
    om, wt = W.omega_grid(cfg.n_omega)
    ptot = int(cfg.n_proj.sum()) if ptot is None else ptot
    return B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, batch, ptot, "cuda:0")


def _dev(kd):
    import torch
    return {k: torch.from_numpy(getattr(kd, k)).to("cuda:0") for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}


def test_empty_band_sets_are_a_no_op_and_reset_zeroes():
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    h = _handle(cfg)
    try:
        kd = W.kpoint(cfg, 0)
        d = _dev(kd)
        empty = torch.empty((0,) + tuple(cfg.grid), dtype=torch.complex128, device="cuda:0")
        B.rpa_chi0_add_kpoint(h, 1.0, empty, d["psi_unocc"], [], kd.eps_unocc, [], kd.f_unocc)
        B.rpa_chi0_add_kpoint(h, 1.0, d["psi_occ"], empty, kd.eps_occ, [], kd.f_occ, [])
        assert float(B.rpa_chi0_get(h, 0).abs().max()) == 0.0
        B.rpa_chi0_add_kpoint(h, 1.0, d["psi_occ"], d["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc)
        assert float(B.rpa_chi0_get(h, 0).abs().max()) > 0.0
        B.rpa_chi0_reset(h)
        for i in range(cfg.n_omega):
            assert float(B.rpa_chi0_get(h, i).abs().max()) == 0.0
    finally:
        h.close()


def test_single_pair_and_single_band_tails():
    """K = 1 (one chunk of 16 pairs, 15 of them padding) and 1 x n / n x 1 band sets against the oracle."""
    from paper_1307_8052_b200 import binding as B
    import torch
    cfg = W.CONFIGS[0]
    for occ, unocc in (([1], [5]), ([0, 2, 3], [7]), ([2], list(range(0, 28, 3)))):
        kd = W.kpoint(cfg, 0, occ=occ, unocc=unocc)
        h = _handle(cfg)
        try:
            g, K2 = B.rpa_chi0_gvectors(h)
            Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
            B.add_kpoint_host(h, kd, cfg.n_proj, Qd, W.atom_positions(cfg))
            chi_g = [B.rpa_chi0_get(h, i).cpu().numpy() for i in range(cfg.n_omega)]
        finally:
            h.close()
        chi_o, _, _, _ = oracle_run(cfg, [kd], True, want_ec=False)
        for i in range(cfg.n_omega):
            assert rel_fro(chi_g[i], chi_o[i]) <= 1e-10


def test_argument_errors_are_reported_not_thrown():
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    h = _handle(cfg, ptot=4)   # room for 4 projectors only
    try:
        kd = W.kpoint(cfg, 0)
        d = _dev(kd)
        g, K2 = B.rpa_chi0_gvectors(h)
        for bad in (-1, cfg.n_omega):
            with pytest.raises(B.RpaError) as ei:
                B.rpa_chi0_get(h, bad)
            assert ei.value.code == B.RPA_ERR_INVALID_ARG
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
        with pytest.raises(B.RpaError) as ei:   # 8 projectors > max_proj_total = 4 given at create
            B.rpa_chi0_add_kpoint(h, 1.0, d["psi_occ"], d["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc,
                                  cfg.n_proj, d["P_occ"], d["P_unocc"], Qd, W.atom_positions(cfg))
        assert ei.value.code == B.RPA_ERR_WORKSPACE
        v = W.coulomb(K2)
        for bad_v in (np.where(np.arange(len(v)) == 3, 0.0, v), np.where(np.arange(len(v)) == 5, np.nan, v), -v):
            with pytest.raises(B.RpaError) as ei:
                B.rpa_ec_q(h, bad_v)
            assert ei.value.code == B.RPA_ERR_INVALID_ARG
        assert "v_G" in B.rpa_last_error()
        # the handle is still usable after the errors
        B.rpa_chi0_add_kpoint(h, 1.0, d["psi_occ"], d["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc)
        ec, e = B.rpa_ec_q(h, v)
        assert np.isfinite(ec) and ec < 0.0
    finally:
        h.close()


def test_not_positive_definite_is_detected():
    """Swapped occupations give positive weights, chi0 >= 0, and I - v^1/2 chi0 v^1/2 loses positive definiteness
    once scaled up: rpa_ec_q must return RPA_ERR_NOT_PD, and chi0 must be left untouched."""
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    h = _handle(cfg, ptot=0)
    try:
        kd = W.kpoint(cfg, 0)
        d = _dev(kd)
        g, K2 = B.rpa_chi0_gvectors(h)
        B.rpa_chi0_add_kpoint(h, 1.0e3, d["psi_occ"], d["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_unocc[:cfg.n_occ] * 0.0,
                              np.ones(cfg.n_unocc))
        before = B.rpa_chi0_get(h, 0).cpu().numpy()
        assert np.linalg.eigvalsh(before).min() >= -1e-10 * np.abs(before).max()
        with pytest.raises(B.RpaError) as ei:
            B.rpa_ec_q(h, W.coulomb(K2))
        assert ei.value.code == B.RPA_ERR_NOT_PD
        assert np.array_equal(B.rpa_chi0_get(h, 0).cpu().numpy(), before)
    finally:
        h.close()


def test_unsupported_grid_length_is_rejected():
    from paper_1307_8052_b200 import binding as B
    cell = np.diag([6.0, 6.5, 7.0])
    om, wt = W.omega_grid(4)
    with pytest.raises(B.RpaError) as ei:   # N3 = 11: prime factor other than 2, 3, 5, 7
        B.rpa_chi0_create((6, 6, 11), cell, (0.25, 0.0, 0.0), 1.0, om, wt, 0, 0, "cuda:0")
    assert ei.value.code == B.RPA_ERR_UNSUPPORTED
    h = B.rpa_chi0_create((11, 6, 8), cell, (0.25, 0.0, 0.0), 1.0, om, wt, 0, 0, "cuda:0")   # N1 is unrestricted
    h.close()


def test_spin_degeneracy_setter():
    """NEXT-4: s = 1 with two different spin channels against the oracle; invalid s is rejected; s scales the read-out."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[0]
    up = W.kpoint(cfg, 0, occ=[0, 1, 2], unocc=range(0, 28, 2))
    dn = W.kpoint(cfg, 0, occ=[1, 3], unocc=range(1, 28, 3))
    h = _handle(cfg, ptot=0)
    try:
        B.rpa_chi0_set_spin_degeneracy(h, 1)
        for kd in (up, dn):
            d = _dev(kd)
            B.rpa_chi0_add_kpoint(h, 1.0, d["psi_occ"], d["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc)
        chi1 = np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(cfg.n_omega)])
        g, K2 = B.rpa_chi0_gvectors(h)
        ec1, _ = B.rpa_ec_q(h, W.coulomb(K2))
        B.rpa_chi0_set_spin_degeneracy(h, 2)
        chi2 = B.rpa_chi0_get(h, 0).cpu().numpy()
        with pytest.raises(B.RpaError) as ei:
            B.rpa_chi0_set_spin_degeneracy(h, 3)
        assert ei.value.code == B.RPA_ERR_INVALID_ARG
    finally:
        h.close()
    import oracle
    om, wt = W.omega_grid(cfg.n_omega)
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, spin_deg=1)
    for kd in (up, dn):
        kd.kweight = 1.0
        orc.add_kpoint(kd)
    chi_o = orc.get()
    for i in range(cfg.n_omega):
        assert rel_fro(chi1[i], chi_o[i]) <= 1e-10
    assert np.allclose(chi2, 2.0 * chi1[0], rtol=1e-15, atol=0)
    ec_o, _ = orc.ec_q(W.coulomb(orc.K2))
    assert abs(ec1 - ec_o) <= 1e-9 * abs(ec_o)
    assert abs(B.rpa_total_energy([ec1, 2 * ec1], [0.25, 0.75]) - 1.75 * ec1) <= 1e-15 * abs(ec1)


def test_ec_q_range_partial_sums_and_isolation():
    """rpa_ec_q_range (reduce-scatter exchange): partial values over disjoint ranges add up to rpa_ec_q,
    e(omega) agrees value by value, a range reads only its own accumulators (the others are poisoned with NaN, as
    they would hold partial sums after a reduce-scatter), invalid ranges are rejected, an empty range gives 0."""
    import torch
    from paper_1307_8052_b200 import binding as B
    from paper_1307_8052_b200 import sharding
    cfg = W.CONFIGS[0]
    h = _handle(cfg)
    try:
        kd = W.kpoint(cfg, 0)
        g, K2 = B.rpa_chi0_gvectors(h)
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
        B.add_kpoint_host(h, kd, cfg.n_proj, Qd, W.atom_positions(cfg))
        v = W.coulomb(K2)
        ec, e = B.rpa_ec_q(h, v)
        for world in (2, 3, cfg.n_omega + 2):
            parts = [B.rpa_ec_q_range(h, v, *sharding.omega_range(cfg.n_omega, r, world)) for r in range(world)]
            assert abs(sum(p[0] for p in parts) - ec) <= 1e-13 * abs(ec)
            assert np.array_equal(np.concatenate([p[1] for p in parts]), e)
        assert B.rpa_ec_q_range(h, v, 3, 3) == (0.0, pytest.approx(np.zeros(0)))
        for lo, hi in ((-1, 2), (0, cfg.n_omega + 1), (5, 4)):
            with pytest.raises(B.RpaError) as ei:
                B.rpa_ec_q_range(h, v, lo, hi)
            assert ei.value.code == B.RPA_ERR_INVALID_ARG
        S = B.rpa_chi0_accumulators(h).view(cfg.n_omega, -1)
        lo, hi = 2, 5
        keep = S[lo:hi].clone()
        S.fill_(complex(float("nan"), float("nan")))
        S[lo:hi] = keep
        torch.cuda.synchronize()
        ec_p, e_p = B.rpa_ec_q_range(h, v, lo, hi)
        assert np.array_equal(e_p, e[lo:hi])
        om, wt = W.omega_grid(cfg.n_omega)
        assert abs(ec_p - float(np.dot(wt[lo:hi], e[lo:hi])) / (2 * np.pi)) <= 1e-14 * abs(ec)
    finally:
        h.close()


def test_ec_q_lanes_give_the_same_numbers():
    """rpa_ec_q factorises the frequencies of a group in 1 ... 4 concurrent lanes (rpa_chi0_set_ec_lanes):
    every matrix goes through the same arithmetic whichever lane it is in, so e(omega) must agree bit for bit, for an
    even split, a ragged one (8 frequencies in 3 lanes) and more lanes than frequencies (a range of 2).  nG = 401
    (configs[2]) spans four 128-column blocks with a ragged last one: look-ahead and big updates both run."""
    import torch
    from paper_1307_8052_b200 import binding as B
    for cfg, n_unocc in ((W.CONFIGS[0], None), (W.CONFIGS[2], 24)):
        h = _handle(cfg)
        try:
            kd = W.kpoint(cfg, 0) if n_unocc is None else W.kpoint(cfg, 0, unocc=range(n_unocc))
            g, K2 = B.rpa_chi0_gvectors(h)
            Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
            B.add_kpoint_host(h, kd, cfg.n_proj, Qd, W.atom_positions(cfg))
            v = W.coulomb(K2)
            ref = None
            # RPA_EC_FLAG_WIDE_TILES: the chain updates in the 64 x 64 tiles of the big updates instead of their own
            # 32 x 32-tile kernel -- the same sums in the same order, so also bit for bit
            for lanes in (1, 2, 3, 4, 2 | B.RPA_EC_FLAG_WIDE_TILES, 3 | B.RPA_EC_FLAG_WIDE_TILES):
                B.rpa_chi0_set_ec_lanes(h, lanes)
                ec, e = B.rpa_ec_q(h, v)
                ec2, e2 = B.rpa_ec_q_range(h, v, 1, 3)
                if ref is None:
                    ref = (ec, e, ec2, e2)
                    assert np.all(np.isfinite(e)) and np.all(e < 0.0)
                else:
                    assert ec == ref[0] and np.array_equal(e, ref[1])
                    assert ec2 == ref[2] and np.array_equal(e2, ref[3])
            for bad in (0, 5, B.RPA_EC_FLAG_WIDE_TILES, 0x200 | 2):
                with pytest.raises(B.RpaError) as ei:
                    B.rpa_chi0_set_ec_lanes(h, bad)
                assert ei.value.code == B.RPA_ERR_INVALID_ARG
        finally:
            h.close()


def test_int8_tcgen05_probe_self_check():
    """rpa_probe_int8_tensor_peak: the TMEM read-back of one tcgen05.mma.kind::i8 equals the host product bit for bit,
    and the issue rate is in the range of a Blackwell int8 tensor pipe (legacy mma.sync reaches 1.1 Pop/s)."""
    from paper_1307_8052_b200 import probes
    tops, bad = probes.rpa_probe_int8_tensor_peak("cuda:0")
    assert bad == 0
    assert 2000.0 < tops < 6000.0
    tf = probes.rpa_probe_fp64_tensor_peak("cuda:0")
    assert 20.0 < tf < 60.0   # B200: 40 TFLOP/s nominal FP64


def test_nothing_is_written_outside_the_workspace_and_the_outputs():
    """A write-bounds check of every kernel of the path (compute-sanitizer is closed on this GPU pool, see
    profiles/r2_sanitizer.md): the workspace, chi0_out and psi_out sit between 8 MB guard bands filled with a byte
    pattern; after add_kpoint (PAW, both FP64 kernels, the int8 kernel with and without clusters, 6 / 7 / 8 digits),
    get, ec_q (Cholesky), pw_to_grid and symmetry_remap on configs[0] and on a ragged skewed-cell grid the bands must be
    untouched and the workspace bytes beyond what rpa_chi0_workspace_bytes reported must be too."""
    import ctypes as C
    import torch
    from paper_1307_8052_b200 import binding as B
    GUARD = 8 << 20

    def guarded(nbytes):
        buf = torch.full((GUARD + nbytes + 256 + GUARD,), 0xA5, dtype=torch.uint8, device="cuda:0")
        off = GUARD + (-(buf.data_ptr() + GUARD)) % 256
        return buf, off

    def check(buf, off, nbytes, what):
        assert bool((buf[:off] == 0xA5).all()), f"{what}: bytes before the buffer were overwritten"
        assert bool((buf[off + nbytes:] == 0xA5).all()), f"{what}: bytes after the buffer were overwritten"

    cell = np.array([[6.0, 0.2, 0.0], [0.1, 5.0, 0.3], [0.0, -0.2, 7.0]])
    ragged = W.custom_config(777, cell, (12, 10, 14), (0.25, 0.0, 0.5), n_occ=3, n_unocc=7, ng_target=33, n_omega=5, n_atoms=2,
                             n_proj_per_atom=3, orb_ecut_ha=2.0)
    modes = [(B.RPA_RANK_K_FP64_3M, 0), (B.RPA_RANK_K_FP64_4M, 0)]
    for digits in (6, 7, 8):
        modes.append((B.RPA_RANK_K_I8 | B.RPA_RANK_K_FLAG_ALL_BATCHES, digits))
    modes.append((B.RPA_RANK_K_I8 | B.RPA_RANK_K_FLAG_ALL_BATCHES | B.RPA_RANK_K_FLAG_NO_CLUSTER, 7))
    for cfg in (W.CONFIGS[0], ragged):
        om, wt = W.omega_grid(cfg.n_omega)
        ptot = int(cfg.n_proj.sum())
        nbytes = B.rpa_chi0_workspace_bytes(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), cfg.n_omega, 48, ptot)
        ws, ws_off = guarded(nbytes)
        g32, c64, q64 = np.asarray(cfg.grid, np.int32), np.ascontiguousarray(cfg.cell, np.float64).reshape(9), np.asarray(cfg.q_red, np.float64)
        out = C.c_void_p()
        stream = torch.cuda.current_stream()
        rc = B.lib().rpa_chi0_create(C.byref(out), g32.ctypes.data_as(C.c_void_p), c64.ctypes.data_as(C.c_void_p),
                                     q64.ctypes.data_as(C.c_void_p), W.tuned_ecut(cfg), cfg.n_omega, om.ctypes.data_as(C.c_void_p),
                                     wt.ctypes.data_as(C.c_void_p), 48, ptot, C.c_void_p(ws.data_ptr() + ws_off), C.c_size_t(nbytes),
                                     C.c_void_p(stream.cuda_stream))
        assert rc == 0, B.rpa_last_error()
        h = B.Handle(out, ws, torch.device("cuda", 0), stream, g32, cfg.n_omega)
        try:
            g, K2 = B.rpa_chi0_gvectors(h)
            ng = len(g)
            kd = W.kpoint(cfg, 0)
            d = _dev(kd)
            Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
            chi_buf, chi_off = guarded(ng * ng * 16)
            chi = chi_buf[chi_off:chi_off + ng * ng * 16].view(torch.complex128).view(ng, ng)
            for mode in modes:
                B.rpa_chi0_set_rank_k_mode(h, *mode)
                B.rpa_chi0_add_kpoint(h, 1.0, d["psi_occ"], d["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc,
                                      cfg.n_proj, d["P_occ"], d["P_unocc"], Qd, W.atom_positions(cfg))
                for i in range(cfg.n_omega):
                    B.rpa_chi0_get(h, i, chi)
                B.rpa_ec_q(h, W.coulomb(K2))
                B.rpa_chi0_sync(h)
                check(ws, ws_off, nbytes, f"workspace, mode {mode}")
                check(chi_buf, chi_off, ng * ng * 16, f"chi0_out, mode {mode}")
            # Table 1 steps 3-4
            g_pw, C_o, _ = W.kpoint_coefficients(cfg, 0, occ=range(cfg.n_occ), unocc=[])
            N = int(np.prod(cfg.grid))
            psi_buf, psi_off = guarded(cfg.n_occ * N * 16)
            psi = psi_buf[psi_off:psi_off + cfg.n_occ * N * 16].view(torch.complex128).view((cfg.n_occ,) + tuple(cfg.grid))
            B.rpa_pw_to_grid(h, g_pw, torch.from_numpy(C_o).to("cuda:0"), psi)
            B.rpa_chi0_sync(h)
            check(psi_buf, psi_off, cfg.n_occ * N * 16, "psi_out of rpa_pw_to_grid")
            check(ws, ws_off, nbytes, "workspace after rpa_pw_to_grid")
            src = psi.clone()
            B.rpa_symmetry_remap(h, src, np.diag([-1, -1, -1]), True, psi)
            B.rpa_chi0_sync(h)
            check(psi_buf, psi_off, cfg.n_occ * N * 16, "psi_out of rpa_symmetry_remap")
        finally:
            h.close()


@pytest.mark.parametrize("ng_target", [20, 33, 64, 97, 129, 160, 257, 300, 385, 520, 777])
def test_ec_q_on_synthetic_accumulators_of_many_sizes(ng_target):
    """The factorisation of rpa_ec_q by itself -- ec_build / ec_trace / chol_panel / the strips and look-ahead columns in
    32 x 32 tiles / the big updates in 64 x 64 tiles -- on spheres whose size sits on and around the panel (32), tile (64)
    and block (128) edges: the accumulators are filled directly with a Hermitian negative semi-definite matrix per frequency
    (skewed cell, no pair densities involved), chi0 is read back with rpa_chi0_get, and e(omega), E_c(q) must agree with the
    oracle's unblocked Cholesky of the same chi0; the lane / tile-shape variants must agree with each other bit for bit."""
    import oracle
    import torch
    from paper_1307_8052_b200 import binding as B
    cell = np.array([[7.0, 0.3, 0.0], [0.2, 7.5, 0.1], [0.0, -0.4, 8.0]])
    cfg = W.custom_config(200 + ng_target, cell, (20, 20, 20), (0.25, 0.1, 0.0), 1, 1, ng_target, 3, 1, 1)
    h = _handle(cfg, ptot=0)
    try:
        ng = B.rpa_chi0_ng(h)
        assert ng == ng_target
        _, K2 = B.rpa_chi0_gvectors(h)
        v = W.coulomb(K2)
        S = B.rpa_chi0_accumulators(h).view(cfg.n_omega, ng, ng)
        rng = np.random.default_rng([77, ng])
        for i in range(cfg.n_omega):
            r = max(1, ng // 3)
            A = (rng.standard_normal((ng, r)) + 1j * rng.standard_normal((ng, r))) / np.sqrt(2.0 * r)
            M = -(A * rng.uniform(0.01, 2.0, r)) @ A.conj().T / np.sqrt(np.outer(v, v))   # v^1/2 chi0 v^1/2 of order one
            M = np.tril(M)                                                                # the library keeps one triangle
            M[np.diag_indices(ng)] = M.diagonal().real
            S[i].copy_(torch.from_numpy(M))
        chi = np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(cfg.n_omega)])
        assert np.array_equal(chi, chi.conj().transpose(0, 2, 1))
        om, wt = W.omega_grid(cfg.n_omega)
        ec_o, e_o = oracle.ec_q(chi, v, wt)
        ref = None
        for lanes in (2, 1, 3, 2 | B.RPA_EC_FLAG_WIDE_TILES):
            B.rpa_chi0_set_ec_lanes(h, lanes)
            ec, e = B.rpa_ec_q(h, v)
            if ref is None:
                ref = (ec, e)
                assert np.all(np.abs(e - e_o) <= 1e-10 * np.abs(e_o)), (e, e_o)
                assert abs(ec - ec_o) <= 1e-10 * abs(ec_o)
            else:
                assert ec == ref[0] and np.array_equal(e, ref[1]), lanes
    finally:
        h.close()
