"""Pins of the NEXT-2 oracle functions: the q -> 0 limit of the G = 0 pair density (Eq. 13)
from gradient matrix elements in the plane-wave basis (Eq. 15 / Eq. 19)."""
import numpy as np

import oracle
from paper_1307_8052_b200 import workload as W


def test_single_plane_waves_closed_form():
    """psi_n = one plane wave each: <n|nabla|m> = i (k + G_n) delta_{G_n G_m}."""
    cell = np.array([[7.0, 0.3, 0.0], [0.0, 6.0, 0.2], [0.1, 0.0, 8.0]])
    B = 2 * np.pi * np.linalg.inv(cell).T
    k = np.array([0.13, -0.07, 0.21])
    g = np.array([[0, 0, 0], [1, 0, -1], [2, 1, 0]])
    C = np.eye(3, dtype=np.complex128)
    G = oracle.momentum_pw(cell, k, g, C, C)
    for al in range(3):
        want = np.diag(1j * (k[al] + (g @ B)[:, al]))
        assert np.abs(G[al] - want).max() < 1e-15


def test_two_plane_wave_mixture_and_antihermiticity():
    """Analytic mixture: n = (|0> + |1>)/sqrt2, m = (|0> - i|1>)/sqrt2 => <n|nabla|m> = i (K0 - i K1)/2; and nabla is
    anti-Hermitian on a common plane-wave set: grad[m][n] = -conj(grad[n][m])."""
    cell = np.diag([6.0, 7.0, 8.0])
    B = 2 * np.pi * np.linalg.inv(cell).T
    k = np.array([0.0, 0.1, 0.2])
    g = np.array([[1, 0, 0], [0, -2, 1]])
    K = k + g @ B
    Cn = np.array([[1, 1]], dtype=np.complex128) / np.sqrt(2)
    Cm = np.array([[1, -1j]], dtype=np.complex128) / np.sqrt(2)
    G = oracle.momentum_pw(cell, k, g, Cn, Cm)
    for al in range(3):
        assert abs(G[al, 0, 0] - 1j * (K[0, al] - 1j * K[1, al]) / 2) < 1e-15
    rng = np.random.default_rng(4)
    gg = rng.integers(-3, 4, (20, 3))
    gg = np.unique(gg, axis=0)
    Ca = rng.standard_normal((3, len(gg))) + 1j * rng.standard_normal((3, len(gg)))
    Cb = rng.standard_normal((4, len(gg))) + 1j * rng.standard_normal((4, len(gg)))
    Gab = oracle.momentum_pw(cell, k, gg, Ca, Cb)
    Gba = oracle.momentum_pw(cell, k, gg, Cb, Ca)
    assert np.abs(Gba + np.conj(Gab.transpose(0, 2, 1))).max() < 1e-13


def test_grid_route_library_special_case():
    """<u_n|(i k + nabla)|u_m> on the grid with a numpy spectral derivative equals the plane-wave sum (config 0)."""
    cfg = W.CONFIGS[0]
    B = 2 * np.pi * np.linalg.inv(cfg.cell).T
    g, C0 = W.orbital_coefficients(cfg, 0, 1)
    _, C1 = W.orbital_coefficients(cfg, 0, 9)
    k = np.array([0.1, 0.2, -0.05])
    G = oracle.momentum_pw(cfg.cell, k, g, [C0], [C1])
    u0, u1 = W.orbital(cfg, 0, 1), W.orbital(cfg, 0, 9)
    F = np.fft.fftn(u1)
    gc = np.stack(np.meshgrid(*[np.fft.fftfreq(n, 1.0 / n) for n in cfg.grid], indexing="ij"), -1) @ B
    for al in range(3):
        du = np.fft.ifftn(1j * (k[al] + gc[..., al]) * F)
        assert abs(G[al, 0, 0] - np.mean(np.conj(u0) * du)) < 1e-14


def test_paw_term_closed_form_and_head():
    """One atom, one projector: the PAW term is conj(p_n) Qgrad_al p_m; head = -i qdir . grad / (eps_m - eps_n),
    zero for a degenerate pair."""
    cell = np.diag([6.0, 6.0, 6.0])
    g = np.array([[0, 0, 0], [1, 0, 0]])
    C = np.array([[1.0, 0.0], [0.0, 1.0]], dtype=np.complex128)
    Po, Pu = np.array([[0.3 - 0.2j]]), np.array([[0.1 + 0.5j], [-0.4j]])
    Qg = np.array([0.7 + 0.1j, -0.2j, 1.1])   # [3][1][1]
    G = oracle.momentum_pw(cell, np.zeros(3), g, C[:1], C, [1], Po, Pu, Qg)
    G0 = oracle.momentum_pw(cell, np.zeros(3), g, C[:1], C)
    for al in range(3):
        for m in range(2):
            assert abs(G[al, 0, m] - G0[al, 0, m] - np.conj(Po[0, 0]) * Qg[al] * Pu[m, 0]) < 1e-15
    qd = np.array([0.6, 0.0, 0.8])
    head = oracle.optical_head([-0.5], [0.25, -0.5], qd, G)
    assert abs(head[0, 0] - (-1j) * (qd @ G[:, 0, 0]) / 0.75) < 1e-15
    assert head[0, 1] == 0.0


def test_head_replaces_only_g0_in_chi0():
    """Chi0Oracle with a head: rows/columns other than G = 0 are those of the plain q = 0 run; the G = 0 diagonal is
    (2/Omega) sum w |head|^2."""
    cell = np.diag([6.0, 6.5, 7.0])
    cfg = W.custom_config(321, cell, (6, 6, 6), (0.0, 0.0, 0.0), n_occ=2, n_unocc=5, ng_target=10, n_omega=3, n_atoms=1,
                          n_proj_per_atom=2, orb_ecut_ha=2.0)
    kd = W.kpoint(cfg, 0)
    om, wt = W.omega_grid(cfg.n_omega)
    a = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    b = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    rng = np.random.default_rng(9)
    head = rng.standard_normal((2, 5)) + 1j * rng.standard_normal((2, 5))
    a.add_kpoint(kd)
    b.add_kpoint(kd, head=head)
    i0 = int(np.flatnonzero((a.g == 0).all(axis=1))[0])
    keep = np.arange(a.ng) != i0
    ca, cb = a.get(), b.get()
    assert np.array_equal(ca[:, keep][:, :, keep], cb[:, keep][:, :, keep])
    for i in range(cfg.n_omega):
        w = np.stack([oracle.weights(kd.eps_occ[n], kd.f_occ[n], kd.eps_unocc, kd.f_unocc, om)[i] for n in range(2)])
        want = 2.0 / oracle.volume(cell) * kd.kweight * np.sum(w * np.abs(head) ** 2)
        assert abs(cb[i, i0, i0] - want) < 1e-13 * abs(want)
