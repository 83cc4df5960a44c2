"""Pins of the NEXT-1 oracle functions: plane-wave coefficients -> grid orbitals (Eq. 10)
and the IBZ -> BZ symmetry remap (Eq. 11), against closed forms, a library special case, brute force and
invariants -- none of them retypes the oracle's own formula."""
import numpy as np
import pytest

import oracle
from paper_1307_8052_b200 import workload as W


def _coords(grid):
    return np.stack(np.meshgrid(*[np.arange(n) for n in grid], indexing="ij"), axis=-1)


def test_single_plane_wave_closed_form():
    """C = delta at Q  =>  u_j = exp(2 pi i Q.j/N) exactly (sign and index order of Eq. 10)."""
    grid = (6, 4, 10)
    j = _coords(grid)
    for Q in ([1, 0, 0], [0, -1, 2], [-2, 1, -4]):
        u = oracle.pw_to_grid(grid, [Q], [1.0 + 0.0j]).reshape(grid)
        want = np.exp(2j * np.pi * (j / np.array(grid)) @ np.array(Q))
        assert np.abs(u - want).max() < 1e-14


def test_library_special_case_inverse_fft_and_parseval():
    """u = N * numpy.fft.ifftn(scatter(C)); (1/N) sum |u|^2 = sum |C|^2; config 0 orbitals are reproduced."""
    cfg = W.CONFIGS[0]
    g, C = W.orbital_coefficients(cfg, 0, 5)
    u = oracle.pw_to_grid(cfg.grid, g, C).reshape(cfg.grid)
    Cg = np.zeros(cfg.grid, dtype=np.complex128)
    Cg[g[:, 0], g[:, 1], g[:, 2]] = C
    assert np.abs(u - np.fft.ifftn(Cg) * cfg.n_grid).max() < 1e-13
    assert abs(np.mean(np.abs(u) ** 2) - np.sum(np.abs(C) ** 2)) < 1e-13
    assert np.abs(u - W.orbital(cfg, 0, 5)).max() < 1e-13


def test_brute_force_and_sampled_points():
    rng = np.random.default_rng(3)
    grid = (5, 3, 4)
    g = np.array([[0, 0, 0], [1, -1, 0], [-2, 1, 1], [2, 0, -1]])
    C = rng.standard_normal((2, 4)) + 1j * rng.standard_normal((2, 4))
    u = oracle.pw_to_grid(grid, g, C)
    x = (_coords(grid) / np.array(grid)).reshape(-1, 3)
    want = np.einsum("bq,jq->bj", C, np.exp(2j * np.pi * x @ g.T))
    assert np.abs(u - want).max() < 1e-14
    pts = np.array([0, 7, 59, 33])
    assert np.array_equal(oracle.pw_to_grid(grid, g, C, pts), u[:, pts])


def test_remap_plane_wave_closed_form_identity_and_time_reversal():
    """u = plane wave g  =>  u(M x) is the plane wave M^T g; identity leaves u; time reversal conjugates."""
    grid = (6, 6, 6)
    rng = np.random.default_rng(5)
    u = rng.standard_normal(grid) + 1j * rng.standard_normal(grid)
    assert np.array_equal(oracle.symmetry_remap(grid, np.eye(3, dtype=int), False, u), u)
    assert np.array_equal(oracle.symmetry_remap(grid, np.eye(3, dtype=int), True, u), np.conj(u))
    M = np.array([[0, -1, 0], [1, 0, 0], [0, 0, 1]])   # fourfold rotation about z
    for gvec in ([1, 0, 0], [2, -1, 1]):
        pw = oracle.pw_to_grid(grid, [gvec], [1.0]).reshape(grid)
        out = oracle.symmetry_remap(grid, M, False, pw)
        want = oracle.pw_to_grid(grid, [M.T @ np.array(gvec)], [1.0]).reshape(grid)
        assert np.abs(out - want).max() < 1e-14


def test_remap_composition_inversion_and_incompatible_grid():
    grid = (4, 4, 8)
    rng = np.random.default_rng(6)
    u = rng.standard_normal((2,) + grid) + 1j * rng.standard_normal((2,) + grid)
    M1 = np.array([[0, 1, 0], [1, 0, 0], [0, 0, -1]])
    M2 = np.array([[-1, 0, 0], [0, 1, 0], [0, 0, 1]])
    a = oracle.symmetry_remap(grid, M2, False, oracle.symmetry_remap(grid, M1, False, u))
    assert np.array_equal(a, oracle.symmetry_remap(grid, M1 @ M2, False, u))   # out(x) = in(M1 M2 x)
    inv = oracle.symmetry_remap(grid, -np.eye(3, dtype=int), False, u)
    want = np.roll(u[:, ::-1, ::-1, ::-1], 1, axis=(1, 2, 3))                   # x -> -x on a periodic grid
    assert np.array_equal(inv, want)
    with pytest.raises(ValueError):   # z <-> x swap needs N1 = N3
        oracle.symmetry_remap(grid, np.array([[0, 0, 1], [0, 1, 0], [1, 0, 0]]), False, u)


def test_remapped_orbitals_give_the_rotated_pair_density():
    """Invariant tying Eq. 11 to Eq. 12: with both orbitals taken at M x, ntilde'(g) = ntilde(M^-T g)."""
    grid = (6, 6, 4)
    rng = np.random.default_rng(8)
    un = rng.standard_normal(grid) + 1j * rng.standard_normal(grid)
    um = rng.standard_normal((1,) + grid) + 1j * rng.standard_normal((1,) + grid)
    M = np.array([[0, 1, 0], [-1, 0, 0], [0, 0, 1]])
    g = np.array([[1, 0, 0], [0, 2, 1], [-1, 1, -1], [2, -2, 0]])
    gm = (np.linalg.inv(M).T @ g.T).T.round().astype(np.int32)
    a = oracle.pair_density(grid, oracle.symmetry_remap(grid, M, False, un), oracle.symmetry_remap(grid, M, False, um), g)
    b = oracle.pair_density(grid, un, um, gm)
    assert np.abs(a - b).max() < 1e-14
