"""rpa_e_omega_noalloc (include/rpa_chi0.h): the integrand e(omega) of Eq. 2 (Table 1 step 12) for one
caller-supplied chi0 matrix, with its factorisation scratch in a fixed file-scope device array of the library instead of
a workspace -- for callers that cannot allocate device memory.  Checked against the existing path (rpa_ec_q's e(omega)
of the same chi0, which the parity tests tie to the oracle) on calls made back to back, against the oracle's own
e(omega) on synthetic matrices up to the maximum size, and for what the header promises about the shared array: stale
contents of a larger or failed call do not leak into the next one, sizes beyond the maximum are refused, and the device's
free memory does not move.

Collected last on purpose (the name sorts after every other test file): the suite runs with -x."""
import numpy as np
import pytest

from paper_1307_8052_b200 import workload as W

pytestmark = pytest.mark.gpu

E_TOL = 1e-9   # the relative tolerance of the path's energies (BASELINE.json north_star; EC_TOL of test_gpu_parity.py)
DEV = "cuda:0"


def _existing_path(cfg, n_k=1):
    """chi0 of every frequency as DEVICE tensors, v_G, and e(omega) of rpa_ec_q -- all from a handle of the library."""
    import torch
    from paper_1307_8052_b200 import binding as B
    om, wt = W.omega_grid(cfg.n_omega)
    ptot = int(cfg.n_proj.sum())
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, ptot, DEV)
    try:
        _, K2 = B.rpa_chi0_gvectors(h)
        Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to(DEV)
        for k in range(n_k):
            B.add_kpoint_host(h, W.kpoint(cfg, k), cfg.n_proj, Qd, W.atom_positions(cfg))
        chi = [B.rpa_chi0_get(h, i).clone() for i in range(cfg.n_omega)]
        v = W.coulomb(K2)
        _, e_ref = B.rpa_ec_q(h, v)
        B.rpa_chi0_sync(h)
    finally:
        h.close()
    return chi, v, e_ref


def _noalloc(chi_list, v, stream=None):
    """One call per matrix, back to back on one stream, no synchronisation in between; e as numpy."""
    import torch
    from paper_1307_8052_b200 import binding as B
    v_d = torch.from_numpy(np.ascontiguousarray(v, dtype=np.float64)).to(DEV)
    e_d = torch.full((len(chi_list),), 12345.0, dtype=torch.float64, device=DEV)
    for i, x in enumerate(chi_list):
        B.rpa_e_omega_noalloc(x, v_d, e_d[i:i + 1], stream)
    torch.cuda.synchronize()
    return e_d.cpu().numpy()


def _close(e, e_ref):
    return np.abs(e - e_ref) <= E_TOL * np.abs(e_ref) + 1e-300


def test_matches_rpa_ec_q_on_consecutive_calls():
    """configs[2] (nG = 401: three full 128-column blocks and a ragged 17-column panel), one k-point, PAW on: the 16
    frequencies as 16 calls in a row, twice.  Every e(omega) within the path's tolerance of rpa_ec_q's, and the second
    round bit-identical to the first (same kernels, same order, one stream)."""
    chi, v, e_ref = _existing_path(W.CONFIGS[2])
    assert chi[0].shape[0] > 3 * 128
    e1 = _noalloc(chi, v)
    e2 = _noalloc(chi, v)
    assert np.all(np.isfinite(e1)) and np.all(e_ref < 0.0)
    assert _close(e1, e_ref).all(), (e1, e_ref)
    assert np.array_equal(e1, e2)


def test_smaller_matrix_after_a_larger_one_and_back():
    """The array keeps the last call's contents: a 155 x 155 problem (configs[0]) right after a 401 x 401 one, then the
    large one again, with no synchronisation between the calls -- each must match its own rpa_ec_q value."""
    import torch
    from paper_1307_8052_b200 import binding as B
    big, v_big, e_big = _existing_path(W.CONFIGS[2])
    small, v_small, e_small = _existing_path(W.CONFIGS[0])
    vb = torch.from_numpy(v_big).to(DEV)
    vs = torch.from_numpy(v_small).to(DEV)
    out = torch.zeros(3, dtype=torch.float64, device=DEV)
    B.rpa_e_omega_noalloc(big[3], vb, out[0:1])
    B.rpa_e_omega_noalloc(small[1], vs, out[1:2])
    B.rpa_e_omega_noalloc(big[3], vb, out[2:3])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    want = np.array([e_big[3], e_small[1], e_big[3]])
    assert _close(got, want).all(), (got, want)
    assert got[0] == got[2]


def _synthetic(ng, seed):
    """A Hermitian negative semi-definite chi0 (as on the imaginary axis) with a Coulomb-like v: 1 - v^1/2 chi0 v^1/2 is
    positive definite with eigenvalues spread over two orders of magnitude."""
    rng = np.random.default_rng([20131307, ng, seed])
    r = max(1, ng // 2)
    A = (rng.standard_normal((ng, r)) + 1j * rng.standard_normal((ng, r))) / np.sqrt(2.0 * r)
    d = np.exp(rng.uniform(np.log(0.01), np.log(3.0), r))
    chi = -(A * d) @ A.conj().T
    chi = 0.5 * (chi + chi.conj().T)
    chi[np.diag_indices(ng)] = chi.diagonal().real
    v = 4.0 * np.pi / rng.uniform(0.05, 6.0, ng)
    return chi, v


@pytest.mark.parametrize("ng", [1, 31, 32, 33, 128, 129, 300, 512])
def test_against_the_oracle_up_to_the_maximum_size(ng):
    """Sizes around the panel (32) and block (128) edges and the maximum (RPA_NOALLOC_MAX_NG = 512) against the oracle's
    e(omega) (oracle.ec_q on the same matrix), two different matrices per size in consecutive calls."""
    import oracle
    import torch
    from paper_1307_8052_b200 import binding as B
    assert B.RPA_NOALLOC_MAX_NG == 512
    mats = [_synthetic(ng, s) for s in (0, 1)]
    want = np.array([oracle.ec_q(x[None], v, np.ones(1))[1][0] for x, v in mats])
    out = torch.zeros(2, dtype=torch.float64, device=DEV)
    for i, (x, v) in enumerate(mats):
        B.rpa_e_omega_noalloc(torch.from_numpy(x).to(DEV), torch.from_numpy(v).to(DEV), out[i:i + 1])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert _close(got, want).all(), (ng, got, want)


def test_upper_triangle_is_not_read_and_input_is_not_modified():
    import torch
    from paper_1307_8052_b200 import binding as B
    x, v = _synthetic(200, 7)
    xd, vd = torch.from_numpy(x).to(DEV), torch.from_numpy(v).to(DEV)
    junk = xd.clone()
    iu = torch.triu_indices(200, 200, offset=1, device=DEV)
    junk[iu[0], iu[1]] = complex(float("nan"), float("nan"))
    keep = junk.clone()
    out = torch.zeros(2, dtype=torch.float64, device=DEV)
    B.rpa_e_omega_noalloc(xd, vd, out[0:1])
    B.rpa_e_omega_noalloc(junk, vd, out[1:2])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.isfinite(got).all() and got[0] == got[1]
    assert torch.equal(torch.view_as_real(junk).isnan(), torch.view_as_real(keep).isnan())
    assert torch.equal(torch.nan_to_num(torch.view_as_real(junk)), torch.nan_to_num(torch.view_as_real(keep)))


def test_sizes_beyond_the_maximum_and_bad_arguments_are_refused():
    import torch
    from paper_1307_8052_b200 import binding as B
    n = B.RPA_NOALLOC_MAX_NG + 1
    x = torch.zeros((n, n), dtype=torch.complex128, device=DEV)
    v = torch.ones(n, dtype=torch.float64, device=DEV)
    e = torch.full((1,), 7.0, dtype=torch.float64, device=DEV)
    with pytest.raises(B.RpaError) as err:
        B.rpa_e_omega_noalloc(x, v, e)
    assert err.value.code == -2 and "RPA_NOALLOC_MAX_NG" in str(err.value) and "513" in str(err.value)
    torch.cuda.synchronize()
    assert float(e.cpu()[0]) == 7.0   # nothing was launched
    L = B.lib()
    assert L.rpa_e_omega_noalloc(None, 4, v.data_ptr(), e.data_ptr(), None) == -1
    assert L.rpa_e_omega_noalloc(x.data_ptr(), 0, v.data_ptr(), e.data_ptr(), None) == -1
    assert L.rpa_e_omega_noalloc(x.data_ptr(), -3, v.data_ptr(), e.data_ptr(), None) == -1


def test_not_positive_definite_gives_nan_and_the_next_call_is_clean():
    """chi0 = +2 with v = 1 makes 1 - v^1/2 chi0 v^1/2 = -1: the pivot test fails and e is NaN (rpa_ec_q would return
    RPA_ERR_NOT_PD); the failure flag lives in the shared array and must not survive into the next call."""
    import oracle
    import torch
    from paper_1307_8052_b200 import binding as B
    ng = 70
    bad = torch.eye(ng, dtype=torch.complex128, device=DEV) * 2.0
    ones = torch.ones(ng, dtype=torch.float64, device=DEV)
    x, v = _synthetic(ng, 3)
    out = torch.zeros(2, dtype=torch.float64, device=DEV)
    B.rpa_e_omega_noalloc(bad, ones, out[0:1])
    B.rpa_e_omega_noalloc(torch.from_numpy(x).to(DEV), torch.from_numpy(v).to(DEV), out[1:2])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.isnan(got[0])
    want = oracle.ec_q(x[None], v, np.ones(1))[1][0]
    assert _close(got[1:], np.array([want])).all(), (got, want)


def test_on_a_side_stream_and_free_memory_does_not_move():
    """The caller's stream is honoured (results land after a long kernel queued before them on that stream), and a hundred
    calls leave cudaMemGetInfo's free byte count where it was: nothing is allocated, by the call or by a lazy load."""
    import torch
    from paper_1307_8052_b200 import binding as B
    x, v = _synthetic(257, 11)
    xd, vd = torch.from_numpy(x).to(DEV), torch.from_numpy(v).to(DEV)
    out = torch.zeros(101, dtype=torch.float64, device=DEV)
    B.rpa_e_omega_noalloc(xd, vd, out[0:1])          # set-up of the device happens here
    torch.cuda.synchronize()
    side = torch.cuda.Stream(device=DEV)
    free0, _ = torch.cuda.mem_get_info(torch.device(DEV))
    with torch.cuda.stream(side):
        for i in range(1, 101):
            B.rpa_e_omega_noalloc(xd, vd, out[i:i + 1], side)
    side.synchronize()
    free1, _ = torch.cuda.mem_get_info(torch.device(DEV))
    got = out.cpu().numpy()
    assert free1 == free0, (free0, free1)
    assert np.isfinite(got[0]) and np.all(got == got[0])
