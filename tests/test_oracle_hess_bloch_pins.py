"""Pins of the two oracle functions added for SURVEY.md §8f NEXT-3 / NEXT-4 — the full Cartesian
Hessian (oracle.eval_hess, blip_oracle_eval_hess in oracle/blip_oracle.c) and the Bloch-phase
complex orbitals (oracle.bloch) — against what the mathematics fixes, not against themselves:

  Hessian  brute-force definition over ALL sites (oracle/blip_brute.py, separate code);
           trace = the Laplacian of blip_oracle_eval; quadratic and bilinear tables, whose
           Hessian is J_a^T J_b + J_b^T J_a in closed form (pins every component and the chain
           rule through J); central differences of oracle GRADIENTS; val / grad unchanged;
  Bloch    k = 0 returns the real channels; |psi|^2 does not depend on k; a constant table is a
           plane wave (grad = i k psi, laplace = -|k|^2 psi: pins the product rule's signs and
           its factor 2); central differences of psi VALUES for a random table;
           psi(r + a_j) = exp(i k . a_j) psi(r) (Bloch's theorem).
"""
import numpy as np
import pytest

import oracle
import workloads
from oracle import blip_brute

TRICLINIC = ((20.0, 0.0, 0.0), (3.0, 19.0, 0.0), (2.0, 2.0, 24.0))
ORTHO = ((17.4, 0.0, 0.0), (0.0, 17.4, 0.0), (0.0, 0.0, 11.2))
SKEW = ((5.0, 0.3, -0.2), (1.1, 4.0, 0.7), (-0.6, 0.9, 6.0))


# ------------------------------------------------------------------------------- Hessian
@pytest.mark.parametrize("grid,lat,spread,seed", [((5, 4, 6), TRICLINIC, 20.0, 3), ((4, 4, 4), ORTHO, 3.0, 4),
                                                  ((7, 5, 9), SKEW, 8.0, 5)])
def test_hessian_equals_brute_force_definition(grid, lat, spread, seed):
    A, c, pos = workloads.small_case(grid, 3, 8, lat, seed=seed, spread=spread)
    val, grad, hess, _ = oracle.eval_hess(A, grid, c, pos)
    bval, bgrad, blap, bhess = blip_brute.eval_brute(A, grid, c, pos, want_hessian=True)
    scale = np.abs(bhess).max()
    for q, (i, j) in enumerate(oracle.HESS_COMPONENTS):
        assert np.abs(hess[:, q, :] - bhess[:, i, j, :]).max() < 1e-12 * scale
        assert np.abs(bhess[:, i, j, :] - bhess[:, j, i, :]).max() < 1e-12 * scale
    assert np.abs(val - bval).max() < 1e-13 * np.abs(bval).max()
    assert np.abs(grad - bgrad).max() < 1e-13 * np.abs(bgrad).max()


@pytest.mark.parametrize("lat", [ORTHO, TRICLINIC, SKEW])
def test_hessian_trace_is_the_laplacian_and_value_gradient_are_unchanged(lat):
    grid = (9, 7, 8)
    A, c, pos = workloads.small_case(grid, 5, 200, lat, seed=11, spread=5.0)
    val, grad, lap, cell = oracle.eval_fast(A, grid, c, pos)
    hval, hgrad, hess, hcell = oracle.eval_hess(A, grid, c, pos)
    assert np.array_equal(val, hval) and np.array_equal(grad, hgrad) and np.array_equal(cell, hcell)
    tr = hess[:, 0] + hess[:, 1] + hess[:, 2]
    assert np.abs(tr - lap).max() <= 1e-13 * np.abs(hess).max()


def test_hessian_of_quadratic_and_bilinear_tables_closed_form():
    """c[k] = k_a k_b on interior cells gives S = t_a t_b (+ 1/3 for a = b), so the grid-space
    Hessian is the constant E_ab + E_ba and Hc[i][j] = J[a][i] J[b][j] + J[b][i] J[a][j]."""
    grid = (10, 9, 11)
    n = np.array(grid, dtype=np.float64)
    k0, k1, k2 = np.meshgrid(*[np.arange(g, dtype=np.float64) for g in grid], indexing="ij")
    ks = (k0, k1, k2)
    pairs = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]
    c = np.stack([ks[a] * ks[b] for a, b in pairs], axis=-1).astype(np.float32)
    rng = np.random.default_rng(7)
    u = (1.0 + rng.random((150, 3)) * (n - 3.0)) / n
    for lat in (TRICLINIC, SKEW, ORTHO):
        A = np.asarray(lat, dtype=np.float64)
        _, _, hess, _ = oracle.eval_hess(A, grid, c, u @ A)
        G = np.linalg.inv(A)
        J = n[:, None] * G.T                       # J[a][i] = n_a G[i][a]
        scale = np.abs(J).max() ** 2
        for ch, (a, b) in enumerate(pairs):
            for q, (i, j) in enumerate(oracle.HESS_COMPONENTS):
                expect = J[a, i] * J[b, j] + J[b, i] * J[a, j]
                assert np.abs(hess[:, q, ch] - expect).max() < 1e-9 * scale, (lat, a, b, i, j)


@pytest.mark.parametrize("lat,grid", [(ORTHO, (8, 8, 6)), (TRICLINIC, (7, 6, 8)), (SKEW, (5, 6, 7))])
def test_hessian_by_central_differences_of_gradients(lat, grid):
    A = np.array(lat, dtype=np.float64)
    rng = np.random.default_rng(34)
    c = rng.standard_normal((*grid, 3)).astype(np.float32)
    h = oracle.spacing(A, grid).min()
    n = np.array(grid, dtype=np.float64)
    u = (rng.integers(0, grid, size=(40, 3)) + 0.2 + 0.6 * rng.random((40, 3))) / n    # away from knots (S''' jumps there)
    pos = u @ A
    _, _, hess, _ = oracle.eval_hess(A, grid, c, pos)
    d = 1e-5 * h
    scale = np.abs(hess).max()
    for j in range(3):
        e = np.zeros(3)
        e[j] = 1.0
        gp = oracle.eval_fast(A, grid, c, pos + d * e)[1]
        gm = oracle.eval_fast(A, grid, c, pos - d * e)[1]
        fd = (gp - gm) / (2 * d)                   # fd[:, i, :] = d grad_i / d r_j
        for q, (a, b) in enumerate(oracle.HESS_COMPONENTS):
            if b == j:
                assert np.abs(fd[:, a, :] - hess[:, q, :]).max() < 1e-7 * scale
            if a == j:
                assert np.abs(fd[:, b, :] - hess[:, q, :]).max() < 1e-7 * scale      # symmetry


def test_hessian_non_finite_position():
    A, c, pos = workloads.small_case((6, 6, 6), 2, 4, SKEW, seed=1)
    pos[2, 1] = np.inf
    val, grad, hess, cell = oracle.eval_hess(A, (6, 6, 6), c, pos)
    assert np.isnan(hess[2]).all() and np.isnan(val[2]).all() and (cell[2] == -1).all()
    assert np.isfinite(np.delete(hess, 2, axis=0)).all()


# ------------------------------------------------------------------------------- Bloch phase
def _case(lat, grid, L, M, seed, spread=3.0):
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=seed, spread=spread)
    k = workloads.kpoints(A, L // 2, seed=seed)
    val, grad, lap, _ = oracle.eval_fast(A, grid, c, pos)
    return A, c, pos, k, val, grad, lap


def test_bloch_zero_k_returns_the_real_channels():
    A, c, pos, k, val, grad, lap = _case(SKEW, (6, 5, 7), 8, 30, seed=2)
    psi, gpsi, lpsi = oracle.bloch(val, grad, lap, np.zeros_like(k), pos)
    assert np.array_equal(psi.real, val[:, 0::2]) and np.array_equal(psi.imag, val[:, 1::2])
    assert np.array_equal(gpsi.real, grad[:, :, 0::2]) and np.array_equal(gpsi.imag, grad[:, :, 1::2])
    assert np.array_equal(lpsi.real, lap[:, 0::2]) and np.array_equal(lpsi.imag, lap[:, 1::2])


def test_bloch_modulus_does_not_depend_on_k():
    A, c, pos, k, val, grad, lap = _case(TRICLINIC, (6, 5, 7), 8, 50, seed=3, spread=20.0)
    psi, _, _ = oracle.bloch(val, None, None, k, pos)
    mod2 = val[:, 0::2] ** 2 + val[:, 1::2] ** 2
    assert np.abs(np.abs(psi) ** 2 - mod2).max() <= 1e-14 * mod2.max()
    psi2, g2, l2 = oracle.bloch(val, None, None, 3.0 * k, pos)
    assert g2 is None and l2 is None
    assert np.abs(np.abs(psi2) - np.abs(psi)).max() <= 1e-14 * np.abs(psi).max()


def test_bloch_constant_table_is_a_plane_wave():
    grid, L, M = (6, 5, 7), 6, 40
    A = np.array(TRICLINIC)
    rng = np.random.default_rng(4)
    kappa = rng.integers(-8, 9, size=L) / 4.0
    c = np.broadcast_to(kappa.astype(np.float32), (*grid, L)).copy()
    pos = (rng.random((M, 3)) - 0.5) * 8.0 @ A
    k = workloads.kpoints(A, L // 2, seed=4)
    val, grad, lap, _ = oracle.eval_fast(A, grid, c, pos)
    psi, gpsi, lpsi = oracle.bloch(val, grad, lap, k, pos)
    amp = kappa[0::2] + 1j * kappa[1::2]
    expect = amp[None, :] * np.exp(1j * (pos @ k.T))
    assert np.abs(psi - expect).max() < 1e-13 * np.abs(amp).max()
    assert np.abs(gpsi - 1j * k.T[None, :, :] * expect[:, None, :]).max() < 1e-11
    assert np.abs(lpsi + (k * k).sum(axis=1)[None, :] * expect).max() < 1e-10


@pytest.mark.parametrize("lat,grid", [(ORTHO, (8, 8, 6)), (TRICLINIC, (7, 6, 8))])
def test_bloch_derivatives_by_central_differences_of_values(lat, grid):
    A = np.array(lat, dtype=np.float64)
    rng = np.random.default_rng(35)
    L = 6
    c = rng.standard_normal((*grid, L)).astype(np.float32)
    k = 4.0 * workloads.kpoints(A, L // 2, seed=9)           # |k| comparable with 1/h: every term of the product rule matters
    h = oracle.spacing(A, grid).min()
    n = np.array(grid, dtype=np.float64)
    u = (rng.integers(0, grid, size=(30, 3)) + 0.2 + 0.6 * rng.random((30, 3))) / n
    pos = u @ A

    def psi_at(p):
        return oracle.bloch(oracle.eval_fast(A, grid, c, p, mode=oracle.VALUE)[0], None, None, k, p)[0]

    val, grad, lap, _ = oracle.eval_fast(A, grid, c, pos)
    psi, gpsi, lpsi = oracle.bloch(val, grad, lap, k, pos)
    d1 = 1e-5 * h
    for x in range(3):
        e = np.zeros(3)
        e[x] = 1.0
        fd = (psi_at(pos + d1 * e) - psi_at(pos - d1 * e)) / (2 * d1)
        assert np.abs(fd - gpsi[:, x, :]).max() < 1e-8 * np.abs(gpsi).max() + 1e-9

    def second_difference(d):
        out = np.zeros_like(lpsi)
        for x in range(3):
            e = np.zeros(3)
            e[x] = 1.0
            out += (psi_at(pos + d * e) - 2 * psi + psi_at(pos - d * e)) / (d * d)
        return out

    d2 = 4e-3 * h
    fd2 = (4.0 * second_difference(d2 / 2) - second_difference(d2)) / 3.0      # Richardson, as for the real Laplacian
    assert np.abs(fd2 - lpsi).max() < 1e-6 * np.abs(lpsi).max()


def test_bloch_theorem_under_lattice_translations():
    A, c, pos, k, val, grad, lap = _case(TRICLINIC, (6, 5, 7), 8, 40, seed=6)
    psi, gpsi, lpsi = oracle.bloch(val, grad, lap, k, pos)
    shift = np.array([2.0, -1.0, 3.0]) @ A
    v2, g2, l2, _ = oracle.eval_fast(A, (6, 5, 7), c, pos + shift)
    psi2, gpsi2, lpsi2 = oracle.bloch(v2, g2, l2, k, pos + shift)
    ph = np.exp(1j * (k @ shift))[None, :]
    assert np.abs(psi2 - ph * psi).max() < 1e-12 * np.abs(psi).max()
    assert np.abs(gpsi2 - ph[:, None, :] * gpsi).max() < 1e-11 * np.abs(gpsi).max()
    assert np.abs(lpsi2 - ph * lpsi).max() < 1e-10 * np.abs(lpsi).max()
