"""Pins of the oracle's complex-frequency route (orc_weights_z, orc_accumulate_z, second
workload: chi0 on the real axis, z = omega + i eta; reading A19).  The paper prints no value for it
(P:L299 only names it), so the pins are analytic continuation onto the imaginary-axis route (pinned on its own by
tests/test_oracle_pins.py), symmetries, the sign of the absorptive part and closed-form frequency integrals.  CPU only.
"""
import numpy as np
import pytest

import oracle
from paper_1307_8052_b200 import workload as W


@pytest.fixture(scope="module")
def small():
    cfg = W.custom_config(77, np.diag([6.0, 6.5, 7.0]), (6, 6, 6), (0.25, 0.0, 0.0), n_occ=2, n_unocc=5, ng_target=8,
                          n_omega=3, n_atoms=1, n_proj_per_atom=2, orb_ecut_ha=2.0)
    return cfg, W.kpoint(cfg, 0)


def _chi(cfg, kd, omega, eta=None):
    o = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), omega, None, eta=eta)
    g, K2 = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
    o.add_kpoint(kd, cfg.n_proj, W.paw_Q(cfg, K2), W.atom_positions(cfg))
    return o.get()


def test_continuation_to_the_imaginary_axis(small):
    """z = 0 + i u is the point i u of the imaginary axis: the complex route (both orderings of Eq. 3, as printed)
    must reproduce the real-weight route of the hot path there.  Catches a wrong sign of either term, a dropped
    reversed ordering, a conjugated weight or a transposed n n^H in orc_accumulate_z."""
    cfg, kd = small
    for u in (0.05, 0.7, 9.0):
        a = _chi(cfg, kd, [0.0], eta=u)[0]
        b = _chi(cfg, kd, [u])[0]
        assert np.abs(a - b).max() <= 1e-14 * np.abs(b).max()


def test_negative_frequency_is_the_adjoint(small):
    """w(-omega + i eta) = conj(w(omega + i eta))  =>  chi0(-omega) = chi0(omega)^H."""
    cfg, kd = small
    chi = _chi(cfg, kd, [0.3, -0.3, 1.1, -1.1], eta=0.04)
    for a, b in ((0, 1), (2, 3)):
        assert np.abs(chi[b] - chi[a].conj().T).max() <= 1e-14 * np.abs(chi[a]).max()
    # and the matrix is genuinely non-Hermitian on the real axis (the adjoint relation is not vacuous)
    assert np.abs(chi[0] - chi[0].conj().T).max() > 1e-3 * np.abs(chi[0]).max()


def test_absorptive_part_is_negative_semidefinite(small):
    """(chi0 - chi0^H)/2i = (2/Omega) sum_p Im w_p n_p n_p^H with Im w_p < 0 for omega > 0, occupied below unoccupied:
    a system in its ground state absorbs.  Catches the sign of eta and of the reversed term."""
    cfg, kd = small
    assert kd.eps_occ.max() < kd.eps_unocc.min() and (kd.f_occ[:, None] > kd.f_unocc[None, :]).all()
    for x in _chi(cfg, kd, [0.2, 0.9, 2.5], eta=0.1):
        ah = (x - x.conj().T) / 2j
        ev = np.linalg.eigvalsh(ah)
        assert ev.max() <= 1e-13 * np.abs(ev).max() and ev.min() < 0.0


def test_single_transition_lorentzian_residue_and_area():
    """One transition of energy D: -Im w(omega + i eta) is a Lorentzian of half-width eta at omega = D minus its
    mirror at -D.  Its value at resonance tends to (f_n - f_m)/eta and its integral over omega in (0, inf) is
    2 (f_n - f_m) atan(D/eta) (elementary antiderivative) -- the spectral weight of the transition."""
    from scipy.integrate import quad
    D, fn, fm = 0.37, 0.9, 0.1
    eta = 1e-4
    w = oracle.weights_z(-0.1, fn, [-0.1 + D], [fm], [D + 1j * eta])[0, 0]
    lorentz_mirror = eta / ((2 * D) ** 2 + eta ** 2)
    assert abs(-w.imag - (fn - fm) * (1.0 / eta - lorentz_mirror)) <= 1e-12 / eta
    assert abs(w.real - (-(fn - fm) * 2 * D / ((2 * D) ** 2 + eta ** 2))) <= 1e-9   # only the mirror term is left
    eta = 0.05
    f = lambda om: -oracle.weights_z(-0.1, fn, [-0.1 + D], [fm], [om + 1j * eta])[0, 0].imag
    area = quad(f, 0.0, D, epsabs=1e-12, epsrel=1e-12)[0] + quad(f, D, np.inf, epsabs=1e-12, epsrel=1e-12)[0]
    assert abs(area - 2 * (fn - fm) * np.arctan(D / eta)) <= 1e-9


def test_static_limit_and_high_frequency_tail(small):
    """omega = 0, eta -> 0 is the static response (real, Hermitian, negative semidefinite), and for omega far above
    every transition chi0(omega) -> -chi0(i omega): both tails are (2/Omega) sum 2 (f_n - f_m) D n n^H / omega^2
    with opposite signs (z^2 = +omega^2 against -omega^2)."""
    cfg, kd = small
    stat = _chi(cfg, kd, [0.0], eta=1e-9)[0]
    assert np.abs(stat - stat.conj().T).max() <= 1e-8 * np.abs(stat).max()
    assert np.linalg.eigvalsh(0.5 * (stat + stat.conj().T)).max() <= 1e-12 * np.abs(stat).max()
    big = 4.0e3
    re = _chi(cfg, kd, [big], eta=1e-9)[0]
    im = _chi(cfg, kd, [big])[0]
    dmax = float((kd.eps_unocc.max() - kd.eps_occ.min()))
    assert np.abs(re + im).max() <= 4.0 * (dmax / big) ** 2 * np.abs(im).max()
