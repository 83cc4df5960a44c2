"""The OPT-IN int8-sliced rank-K update (csrc/rank_k_i8.cuh: tcgen05.mma.kind::i8 on digit slices of the FP64
operands, rpa_chi0_set_rank_k_mode(h, RPA_RANK_K_I8 | flags, digits)) against the CPU oracle, through the C ABI.

The library's default is the FP64 tensor kernel; the int8 kernel is selected per handle.  Its contract
(include/rpa_chi0.h) is an ABSOLUTE error bound per element on the scale of the operand rows' power-of-two maxima,
    |dS[g][g']| <= (digits + 2) 2^(-7 digits) sL_g sR_g'(omega) K',
which `test_element_bound_*` checks for EVERY element of the lower triangle -- including rows whose transitions span
twelve orders of magnitude, where that bound is far wider than FP64 rounding (the reason it is not the default).  The
remaining tests: relative Frobenius parity on ordinary inputs for 6 / 7 / 8 digits, ragged tiles and batches, the
s32-exactness guard (fallback to FP64 beyond 37 448 transitions per batch), NaN / Inf propagation, subnormal rows, and
agreement with the FP64 kernel at configs[1] full size.  RPA_RANK_K_FLAG_ALL_BATCHES forces the kernel onto the small
problems the oracle can check element by element."""
import numpy as np
import pytest

from paper_1307_8052_b200 import workload as W
from tests.parity_util import gpu_run, oracle_run, rel_fro

pytestmark = pytest.mark.gpu

CHI_TOL, EC_TOL = 1e-10, 1e-9   # BASELINE.json north_star
U = 2.0 ** -53


def _i8(digits, cluster=True):
    from paper_1307_8052_b200 import binding as B
    mode = B.RPA_RANK_K_I8 | B.RPA_RANK_K_FLAG_ALL_BATCHES
    if not cluster:
        mode |= B.RPA_RANK_K_FLAG_NO_CLUSTER
    return (mode, digits)


@pytest.mark.parametrize("digits,bound", [(8, 2e-14), (7, 2e-13), (6, 3e-11)])
def test_config0_relative_frobenius(digits, bound):
    """155 G vectors (two ragged 128-row blocks per half, three 64-column blocks), 4 x 28 transitions, PAW on: relative
    Frobenius distance from the oracle per frequency inside the path's tolerance and inside what the digit count gives."""
    cfg = W.CONFIGS[0]
    kds = [W.kpoint(cfg, 0)]
    info = {}
    chi, ec, _, _ = gpu_run(cfg, kds, True, 0, want_ec=True, rank_k_mode=_i8(digits), info=info)
    assert info["rank_k_batches"][0] == 0 and info["rank_k_batches"][1] >= 1   # the int8 kernel really ran
    chi_o, ec_o, _, _ = oracle_run(cfg, kds, True)
    for i in range(cfg.n_omega):
        err = rel_fro(chi[i], chi_o[i])
        assert err <= min(CHI_TOL, bound), (i, err)
        assert np.array_equal(chi[i], chi[i].conj().T)
    assert abs(ec[0] - ec_o[0]) <= EC_TOL * abs(ec_o[0])


def _pow2_above(m):
    """2^e with 2^e > m elementwise (1 where m == 0): the row scales of the slicing passes, recomputed here."""
    mant, ex = np.frexp(m)            # m = mant 2^ex, mant in [0.5, 1)  ->  2^ex > m
    return np.where(m > 0, np.ldexp(1.0, ex), 1.0)


def _element_bound_case(cfg, kd, digits, use_paw=True):
    """Every element of the lower triangle of every frequency: |S_gpu - S_oracle| against the header's bound, with the
    row scales recomputed from the ORACLE's pair densities and weights (one batch: all pairs of kd), plus the rounding
    slack of the two FP64 summations being compared (oracle rank-1 sums, GPU recombination): 8 K u sum_p |w||n||n'|.
    Returns max over elements of (error / int8 bound) and of (error / pure FP64 rounding slack)."""
    import oracle
    om, wt = W.omega_grid(cfg.n_omega)
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    Q = R = npj = None
    if use_paw:
        Q, R, npj = W.paw_Q(cfg, orc.K2), W.atom_positions(cfg), cfg.n_proj
    n_occ = kd.psi_occ.shape[0]
    N = np.concatenate([orc.pair_densities(n, kd, npj, Q, R) for n in range(n_occ)])            # [pairs][ng]
    w = np.concatenate([oracle.weights(kd.eps_occ[n], kd.f_occ[n], kd.eps_unocc, kd.f_unocc, om) for n in range(n_occ)],
                       axis=1) * kd.kweight                                                         # [nw][pairs]
    K = N.shape[0]
    Kp = 2 * ((K + 31) // 32 * 32)
    comp = np.maximum(np.abs(N.real), np.abs(N.imag))                                              # [pairs][ng]
    sL = _pow2_above(comp.max(axis=0))                                                             # [ng]
    info = {}
    chi, _, _, _ = gpu_run(cfg, [kd], use_paw, 0, want_ec=False, rank_k_mode=_i8(digits) if digits else None, info=info)
    if digits:
        assert info["rank_k_batches"] == (0, 1)
    chi_o, _, _, _ = oracle_run(cfg, [kd], use_paw, want_ec=False)
    pref = 2.0 / oracle.volume(cfg.cell)
    tril = np.tril(np.ones((orc.ng, orc.ng), dtype=bool))
    worst_i8 = worst_fp = 0.0
    for i in range(cfg.n_omega):
        sR = _pow2_above((np.abs(w[i])[:, None] * comp).max(axis=0))                               # [ng]
        # the pair densities themselves carry the FFT's rounding, absolute on the scale of each pair's largest coefficient
        absN = np.abs(N) + 64.0 * U * np.abs(N).max(axis=1, keepdims=True)
        mag = (absN * np.abs(w[i])[:, None]).T @ absN                                              # sum_p |w||n_g||n_g'|, symmetric
        slack = 8.0 * K * U * mag
        err = np.abs(chi[i] - chi_o[i]) / pref
        if digits:
            bound = (digits + 2) * 2.0 ** (-7 * digits) * np.outer(sL, sR) * Kp
            # factor 2: the library's N differs from the oracle's by rounding, which can move a row maximum across a power of two
            ok = err <= 2.0 * bound + slack
            assert ok[tril].all(), (i, float((err / (2.0 * bound + slack))[tril].max()))
            worst_i8 = max(worst_i8, float((err / bound)[tril].max()))
        else:
            assert (err <= slack)[tril].all(), (i, float((err / slack)[tril].max()))
        worst_fp = max(worst_fp, float((err / slack)[tril].max()))
    return worst_i8, worst_fp


@pytest.mark.parametrize("digits", [0, 6, 7, 8])
def test_element_bound_ordinary_rows(digits):
    """configs[0] as generated: all transitions of a row have comparable size.  digits = 0: the default FP64 kernel, every
    element within the rounding of an FP64 sum of its own terms (8 K u sum_p |w| |n_g| |n_g'|)."""
    cfg = W.CONFIGS[0]
    _element_bound_case(cfg, W.kpoint(cfg, 0), digits)


@pytest.mark.parametrize("digits", [0, 6, 7, 8])
def test_element_bound_rows_spanning_twelve_orders_of_magnitude(digits):
    """One unoccupied orbital is 10^6 times larger than the rest (so its pair densities are, in every row G), and its
    occupation is 1 - 10^-12 so that its weighted contribution w n n' is again comparable to the others' -- the shape of
    the optical-limit head n(G=0) ~ 1/(eps_m - eps_n) of a near-degenerate pair, whose weight ~ (eps_m - eps_n) is tiny.
    FP64 (digits = 0: the default kernel) keeps 53 bits of EVERY term; the int8 slices keep 6 + 7 (digits - 1) bits of
    the row maximum, i.e. 20 bits fewer of the ordinary terms.  The int8 bound must hold element by element; the FP64
    kernel must stay inside pure rounding on the same input."""
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    kd.psi_unocc[5] *= 1.0e6
    kd.P_unocc[5] *= 1.0e6
    kd.f_unocc[5] = 1.0 - 1.0e-12
    worst_i8, worst_fp = _element_bound_case(cfg, kd, digits)
    if digits == 0:
        assert worst_fp <= 1.0
    elif digits <= 7:
        # the point of the case: on such rows the int8 result is far outside FP64 rounding (the bound is what holds)
        assert worst_fp > 10.0, worst_fp


@pytest.mark.parametrize("batch", [16, 48])
def test_small_batches_two_kpoints_no_paw(batch):
    """K = 16 / 48 pairs per batch (one or two 32-pair K blocks per half, zero-padded rows), two k-points."""
    cfg = W.CONFIGS[0]
    kds = [W.kpoint(cfg, 0, occ=[0, 2, 3], unocc=range(0, 28, 2)), W.kpoint(cfg, 1, occ=[1], unocc=range(3, 26))]
    chi, _, _, _ = gpu_run(cfg, kds, False, batch, want_ec=False, rank_k_mode=_i8(7))
    chi_o, _, _, _ = oracle_run(cfg, kds, False, want_ec=False)
    for i in range(cfg.n_omega):
        assert rel_fro(chi[i], chi_o[i]) <= 1e-12


@pytest.mark.parametrize("cluster", [True, False])
def test_config2_ragged_blocks_with_and_without_clusters(cluster):
    """401 G vectors of config 2 (ragged last row / column blocks; with clusters the odd tile rows get a padding tile)."""
    cfg = W.CONFIGS[2]
    kds = [W.kpoint(cfg, 0, occ=[0, 3, 7], unocc=range(0, 300, 7))]
    chi, ec, _, _ = gpu_run(cfg, kds, True, 0, want_ec=True, rank_k_mode=_i8(7, cluster))
    chi_o, ec_o, _, _ = oracle_run(cfg, kds, True)
    for i in range(cfg.n_omega):
        assert rel_fro(chi[i], chi_o[i]) <= 1e-12
    assert abs(ec[0] - ec_o[0]) <= EC_TOL * abs(ec_o[0])


def test_exactness_guard_falls_back_to_fp64_for_huge_batches():
    """The s32 accumulators are provably exact only while digits * 2 Kpad * 64^2 < 2^31.  With max_batch_pairs = 65536
    a batch of 16 x 2400 = 38 400 transitions exceeds the limit for 7 digits (37 448): the library must run the FP64
    kernel for it (rpa_chi0_rank_k_batches says which ran), while 6 digits (limit 43 690) stays on the int8 kernel; both
    must match the oracle."""
    cell = np.eye(3) * 8.0
    cfg = W.custom_config(300, cell, (16, 16, 16), (0.25, 0.0, 0.0), n_occ=16, n_unocc=2400, ng_target=150, n_omega=3,
                          n_atoms=0, n_proj_per_atom=0)
    kds = [W.kpoint(cfg, 0)]
    chi_o, _, _, _ = oracle_run(cfg, kds, False, want_ec=False)
    for digits, want in ((7, (1, 0)), (6, (0, 1))):
        info = {}
        chi, _, _, _ = gpu_run(cfg, kds, False, 65536, want_ec=False, rank_k_mode=_i8(digits), info=info)
        assert info["rank_k_batches"] == want, (digits, info)
        for i in range(cfg.n_omega):
            assert rel_fro(chi[i], chi_o[i]) <= (1e-13 if digits == 7 else 3e-11)


def _run_modes(cfg, kd, Q, modes):
    """chi0 of all frequencies (numpy) from one handle per mode; Q: host array or None."""
    import torch
    from paper_1307_8052_b200 import binding as B
    om, wt = W.omega_grid(cfg.n_omega)
    out = []
    for mode in modes:
        h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, int(cfg.n_proj.sum()), "cuda:0")
        try:
            if mode is not None:
                B.rpa_chi0_set_rank_k_mode(h, *mode)
            Qd = None if Q is None else torch.from_numpy(Q).to("cuda:0")
            B.add_kpoint_host(h, kd, cfg.n_proj if Q is not None else None, Qd, W.atom_positions(cfg))
            out.append(np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(cfg.n_omega)]))
            B.rpa_chi0_sync(h)
        finally:
            h.close()
    return out


@pytest.mark.parametrize("poison", [float("nan"), float("inf")])
def test_non_finite_inputs_propagate_like_the_fp64_kernel(poison):
    """A NaN (or Inf) in Q^a_ij(q+G) at ONE G makes n_p(G) non-finite for every transition: row and column G of chi0 must
    come back non-finite and everything else untouched -- from the int8 kernel exactly as from the FP64 kernel (fmax and
    float -> int conversions silently drop NaNs unless the slicing passes carry them)."""
    import oracle
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    g, K2 = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
    ng = len(g)
    Q = W.paw_Q(cfg, K2)
    g_bad = 77
    Q[(0 * 4 + 1) * ng + g_bad] = poison   # atom 0, (i, j) = (0, 1)
    fp, i8 = _run_modes(cfg, kd, Q, [None, _i8(7)])
    mask = np.zeros((ng, ng), dtype=bool)
    mask[g_bad, :] = mask[:, g_bad] = True
    for i in range(cfg.n_omega):
        assert not np.isfinite(fp[i][mask]).any() and np.isfinite(fp[i][~mask]).all()
        assert not np.isfinite(i8[i][mask]).any() and np.isfinite(i8[i][~mask]).all()
        assert np.abs(i8[i][~mask] - fp[i][~mask]).max() <= 1e-12 * np.abs(fp[i][~mask]).max()


def test_nan_weight_poisons_every_element_in_both_kernels():
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    kd.eps_unocc[2] = float("nan")
    fp, i8 = _run_modes(cfg, kd, None, [None, _i8(7)])
    assert np.isnan(fp).all() and np.isnan(i8).all()


def test_subnormal_rows_stay_finite():
    """Orbitals scaled by 1e-160: every pair density is subnormal (~1e-320), so a row's power-of-two scale would be
    2^1060: the slicing pass clamps the exponent instead of producing inf (and 0 * inf = NaN).  chi0 underflows to 0 in
    both kernels."""
    cfg = W.CONFIGS[0]
    kd = W.kpoint(cfg, 0)
    kd.psi_occ *= 1e-160
    kd.psi_unocc *= 1e-160
    fp, i8 = _run_modes(cfg, kd, None, [None, _i8(7)])
    assert np.isfinite(i8).all() and np.isfinite(fp).all()
    assert np.abs(i8).max() == 0.0 and np.abs(fp).max() == 0.0


def test_int8_and_fp64_kernels_agree_at_full_size():
    """configs[1], all 7200 transitions, device-resident: the int8 kernel as the library would pick it for large batches
    (no ALL_BATCHES flag: nG = 1200, K = 3600 are above its thresholds), 7 and 8 digits, against the default FP64 tensor
    kernel on the whole matrices; both are checked against the oracle elsewhere (tests/test_gpu_parity.py)."""
    import torch
    from paper_1307_8052_b200 import binding as B
    cfg = W.CONFIGS[1]
    kd = W.kpoint(cfg, 0)
    om, wt = W.omega_grid(cfg.n_omega)
    dv = {k: torch.from_numpy(getattr(kd, k)).to("cuda:0") for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
    out = {}
    for mode in ("fp64", "i8x7", "i8x8"):
        h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, int(cfg.n_proj.sum()), "cuda:0")
        try:
            if mode != "fp64":
                B.rpa_chi0_set_rank_k_mode(h, B.RPA_RANK_K_I8, int(mode[-1]))
            g, K2 = B.rpa_chi0_gvectors(h)
            Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to("cuda:0")
            B.rpa_chi0_set_profiling(h, True)
            B.rpa_chi0_add_kpoint(h, kd.kweight, dv["psi_occ"], dv["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ, kd.f_unocc,
                                  cfg.n_proj, dv["P_occ"], dv["P_unocc"], Qd, W.atom_positions(cfg))
            B.rpa_chi0_sync(h)
            ms, n = B.rpa_chi0_stage_times(h)
            assert (n[5] > 0) == (mode != "fp64")   # the kernel that ran is the one the mode names
            fp_b, i8_b = B.rpa_chi0_rank_k_batches(h)
            assert (fp_b, i8_b) == ((1, 0) if mode == "fp64" else (0, 1))   # 12 x 600 transitions: one batch
            out[mode] = ([B.rpa_chi0_get(h, i).cpu().numpy() for i in (0, 7, 15)], B.rpa_ec_q(h, W.coulomb(K2))[0])
        finally:
            h.close()
    for mode, tol in (("i8x7", 2e-13), ("i8x8", 2e-14)):
        for a, b in zip(out[mode][0], out["fp64"][0]):
            assert rel_fro(a, b) <= tol, (mode, rel_fro(a, b))
        assert abs(out[mode][1] - out["fp64"][1]) <= 1e-13 * abs(out["fp64"][1])
