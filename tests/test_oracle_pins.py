"""Pins of the CPU fp64 oracle (oracle/blip_oracle.c) against what the paper and the
mathematics fix — none of them re-types the oracle's own formulas.

Paper: psi_l(r) = sum_{s=1..64} a_ls Theta_s(r), Theta_s a tensor product of a compact 1-D
polynomial with 4 non-zero sites per axis (Eq. 6-7), the 64 sites a subset
of the whole periodic grid (Eq. 8).  Readings: DESIGN.md "Readings".

Each test is aimed at a plausible mistake:
  brute force ........ wrong weight polynomial, wrong site offset (i-1..i+2), wrong wrap,
                       wrong table stride / transposed axes, wrong metric mapping
  partition of unity . normalisation (R2)
  ramps / moments .... dropped or mis-signed derivative term, wrong J / Q = J J^T
  knot values ........ (tests/golden/knot_values.txt) value at sites, site <-> index (R4)
  cosine ............. periodic wrap across the seam
  periodicity ........ triclinic inverse lattice
  finite differences . gradient / Laplacian as derivatives of the oracle's VALUES
  scipy BSpline ...... the 1-D factor against a library routine
  cell index ......... adversarial inputs for the pinned fp64 index map
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
import workloads
from oracle import blip_brute

TRICLINIC = ((20.0, 0.0, 0.0), (3.0, 19.0, 0.0), (2.0, 2.0, 24.0))
ORTHO = ((17.4, 0.0, 0.0), (0.0, 17.4, 0.0), (0.0, 0.0, 11.2))
SKEW = ((5.0, 0.3, -0.2), (1.1, 4.0, 0.7), (-0.6, 0.9, 6.0))
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "knot_values.txt")


def golden():
    out = {}
    with open(GOLDEN) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            name, num, den = line.split()
            out[name] = Fraction(int(num), int(den))
    return out


def frac_to_cart(A, u):
    return np.asarray(u, dtype=np.float64) @ np.asarray(A, dtype=np.float64)


# ----------------------------------------------------------------------------------------
# 1. the definition, summed over ALL sites (separate code: oracle/blip_brute.py)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("grid,lat,spread,seed", [
    ((5, 4, 6), TRICLINIC, 50.0, 3),
    ((4, 4, 4), ORTHO, 3.0, 4),
    ((7, 5, 9), SKEW, 8.0, 5),
    ((4, 9, 5), TRICLINIC, 1.0, 6),
])
def test_fast_equals_brute_force(grid, lat, spread, seed):
    A, c, pos = workloads.small_case(grid, 5, 24, lat, seed=seed, spread=spread)
    val, grad, lap, _ = oracle.eval_fast(A, grid, c, pos)
    bval, bgrad, blap = blip_brute.eval_brute(A, grid, c, pos)
    J = np.array(grid)[:, None] * np.linalg.inv(A).T          # scale of d/dr
    s1 = np.abs(J).max()
    assert np.abs(val - bval).max() < 1e-12
    assert np.abs(grad - bgrad).max() < 1e-12 * s1
    assert np.abs(lap - blap).max() < 1e-11 * s1 * s1


def test_value_mode_equals_vgl_value():
    A, c, pos = workloads.small_case((6, 7, 5), 4, 40, SKEW, seed=11)
    v0, g0, l0, cell0 = oracle.eval_fast(A, (6, 7, 5), c, pos, mode=oracle.VALUE)
    v1, _, _, cell1 = oracle.eval_fast(A, (6, 7, 5), c, pos, mode=oracle.VGL)
    assert g0 is None and l0 is None
    assert np.array_equal(v0, v1) and np.array_equal(cell0, cell1)


# ----------------------------------------------------------------------------------------
# 2. normalisation: partition of unity (reading R2)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("lat", [ORTHO, TRICLINIC])
def test_partition_of_unity(lat):
    grid, L = (9, 6, 7), 3
    kappa = np.array([1.0, -2.5, 1024.0], dtype=np.float32)
    c = np.broadcast_to(kappa, (*grid, L)).copy()
    pos = frac_to_cart(lat, (np.random.default_rng(0).random((200, 3)) - 0.5) * 7.0)
    val, grad, lap, _ = oracle.eval_fast(lat, grid, c, pos)
    assert np.abs(val - kappa[None, :]).max() <= 1e-14 * 1024   # 64-term fp64 sum
    assert np.abs(grad).max() <= 1e-12 * 1024
    assert np.abs(lap).max() <= 1e-11 * 1024


# ----------------------------------------------------------------------------------------
# 3. closed forms from the moment identities of the cubic B-spline, interior cells only
#    sum_k B(t-k) = 1, sum_k k B = t, sum_k k^2 B = t^2 + 1/3, sum_k k^3 B = t^3 + t
# ----------------------------------------------------------------------------------------
def _interior_positions(A, grid, axis, M, seed):
    """positions whose 4 sites along `axis` do not wrap: t_axis in [1, n-2)."""
    rng = np.random.default_rng(seed)
    u = rng.random((M, 3))
    n = grid[axis]
    u[:, axis] = (1.0 + u[:, axis] * (n - 3.0)) / n
    return u, frac_to_cart(A, u)


@pytest.mark.parametrize("lat", [ORTHO, TRICLINIC, SKEW])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_polynomial_coefficients_closed_form(lat, axis):
    grid = (11, 12, 13)
    n = np.array(grid, dtype=np.float64)
    k = np.arange(grid[axis], dtype=np.float64)
    shape = [1, 1, 1]
    shape[axis] = grid[axis]
    kk = np.broadcast_to(k.reshape(shape), grid)
    alpha, beta = 0.75, -1.5
    # exactly representable fp32 coefficients (small integers and dyadic fractions)
    c = np.stack([alpha + beta * kk, kk ** 2, kk ** 3], axis=-1).astype(np.float32)
    u, pos = _interior_positions(lat, grid, axis, 300, seed=axis)
    val, grad, lap, _ = oracle.eval_fast(lat, grid, c, pos)
    t = u[:, axis] * n[axis]
    G = np.linalg.inv(np.asarray(lat, dtype=np.float64))
    Ja = n[axis] * G[:, axis]                  # d t_axis / d r_i
    Qaa = Ja @ Ja
    # linear ramp: S = alpha + beta t, grad = beta dt/dr, lap = 0
    assert np.abs(val[:, 0] - (alpha + beta * t)).max() < 1e-12
    assert np.abs(grad[:, :, 0] - beta * Ja[None, :]).max() < 1e-12 * np.abs(Ja).max() * 10
    assert np.abs(lap[:, 0]).max() < 1e-10 * Qaa
    # quadratic: S = t^2 + 1/3, grad = 2 t dt/dr, lap = 2 Q_aa
    assert np.abs(val[:, 1] - (t ** 2 + 1.0 / 3.0)).max() < 1e-11
    assert np.abs(grad[:, :, 1] - (2 * t)[:, None] * Ja[None, :]).max() < 1e-10
    assert np.abs(lap[:, 1] - 2.0 * Qaa).max() < 1e-10 * Qaa
    # cubic: S = t^3 + t, grad = (3 t^2 + 1) dt/dr, lap = 6 t Q_aa
    assert np.abs(val[:, 2] - (t ** 3 + t)).max() < 1e-9
    assert np.abs(grad[:, :, 2] - (3 * t ** 2 + 1)[:, None] * Ja[None, :]).max() < 1e-9
    assert np.abs(lap[:, 2] - 6.0 * t * Qaa).max() < 1e-9 * Qaa


def test_bilinear_coefficients_pin_the_cross_terms():
    """c[k] = k_a k_b  =>  S = t_a t_b, so the Laplacian is 2 Q[a][b]: non-zero only for a
    non-orthogonal lattice — pins the off-diagonal (mixed second derivative) terms."""
    grid = (10, 9, 11)
    n = np.array(grid, dtype=np.float64)
    k0, k1, k2 = np.meshgrid(*[np.arange(g, dtype=np.float64) for g in grid], indexing="ij")
    c = np.stack([k0 * k1, k0 * k2, k1 * k2], axis=-1).astype(np.float32)
    rng = np.random.default_rng(7)
    u = (1.0 + rng.random((200, 3)) * (n - 3.0)) / n
    for lat in (TRICLINIC, SKEW, ORTHO):
        pos = frac_to_cart(lat, u)
        val, grad, lap, _ = oracle.eval_fast(lat, grid, c, pos)
        G = np.linalg.inv(np.asarray(lat, dtype=np.float64))
        J = n[:, None] * G.T
        Q = J @ J.T
        t = u * n
        for ch, (a, b) in enumerate([(0, 1), (0, 2), (1, 2)]):
            assert np.abs(val[:, ch] - t[:, a] * t[:, b]).max() < 1e-11
            g_expect = t[:, b, None] * J[a][None, :] + t[:, a, None] * J[b][None, :]
            assert np.abs(grad[:, :, ch] - g_expect).max() < 1e-10
            assert np.abs(lap[:, ch] - 2.0 * Q[a, b]).max() < 1e-9 * max(1.0, np.abs(Q).max())


# ----------------------------------------------------------------------------------------
# 4. knot values (tests/golden/knot_values.txt): unit impulse at site k0
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("k0", [(3, 4, 2), (0, 0, 0), (7, 6, 8)])
def test_impulse_knot_values(k0):
    gold = golden()
    grid = (8, 7, 9)
    c = np.zeros((*grid, 1), dtype=np.float32)
    c[k0] = 1.0
    n = np.array(grid)

    def at(offset):
        u = ((np.array(k0) + np.array(offset)) % n) / n
        val, _, _, cell = oracle.eval_fast(TRICLINIC, grid, c, frac_to_cart(TRICLINIC, u)[None])
        return val[0, 0]

    assert abs(at((0, 0, 0)) - float(gold["site_itself"])) < 1e-15
    for off in [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]:
        assert abs(at(off) - float(gold["face_neighbour"])) < 1e-15
    for off in [(1, 1, 0), (-1, 0, 1), (0, -1, -1)]:
        assert abs(at(off) - float(gold["edge_neighbour"])) < 1e-15
    for off in [(1, 1, 1), (-1, 1, -1)]:
        assert abs(at(off) - float(gold["corner_neighbour"])) < 1e-15
    for off in [(2, 0, 0), (0, -2, 0), (0, 0, 2), (3, 1, 1)]:
        assert abs(at(off) - float(gold["two_sites_away"])) < 1e-15


def test_one_dimensional_knot_derivatives():
    """c = delta(k_a, k0) on one axis, constant on the others: S = B(t_a - k0).  At the knots
    B' = +1/2, 0, -1/2 and B'' = 1, -2, 1 (golden file)."""
    gold = golden()
    grid = (8, 8, 8)
    lat = ((8.0, 0, 0), (0, 8.0, 0), (0, 0, 8.0))          # unit spacing: d/dr = d/dt
    for axis in range(3):
        c = np.zeros((*grid, 1), dtype=np.float32)
        idx = [slice(None)] * 3
        idx[axis] = 4
        c[tuple(idx)] = 1.0
        for dt, dname, d2name in [(-1, "dB_at_minus1", "d2B_at_1"), (0, "dB_at_0", "d2B_at_0"),
                                  (1, "dB_at_plus1", "d2B_at_1")]:
            r = np.array([0.3, 0.3, 0.3])
            r[axis] = 4.0 + dt
            val, grad, lap, _ = oracle.eval_fast(lat, grid, c, r[None])
            assert abs(val[0, 0] - float(gold["B_1"] if dt else gold["B_0"])) < 1e-15
            assert abs(grad[0, axis, 0] - float(gold[dname])) < 1e-15
            other = [a for a in range(3) if a != axis]
            assert np.abs(grad[0, other, 0]).max() < 1e-15
            assert abs(lap[0, 0] - float(gold[d2name])) < 1e-14


# ----------------------------------------------------------------------------------------
# 5. discrete cosine eigenfunction across the periodic seam
#    c[k] = cos(2 pi m k / n)  =>  S(grid point k) = cos(2 pi m k / n) (2 + cos(2 pi m / n)) / 3
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("axis,m", [(0, 1), (1, 2), (2, 3)])
def test_cosine_eigenfunction_at_grid_points(axis, m):
    grid = (9, 10, 11)
    n = grid[axis]
    k = np.arange(n)
    shape = [1, 1, 1]
    shape[axis] = n
    cos = np.cos(2 * np.pi * m * k / n).astype(np.float32)
    c = np.broadcast_to(cos.reshape(shape), grid)[..., None].copy()
    u = np.full((n, 3), 0.37)
    u[:, axis] = k / n
    val, _, _, cell = oracle.eval_fast(SKEW, grid, c, frac_to_cart(SKEW, u))
    km = np.roll(cos.astype(np.float64), 1)
    kp = np.roll(cos.astype(np.float64), -1)
    # exact for the fp32-rounded coefficients: (c[k-1] + 4 c[k] + c[k+1]) / 6
    assert np.abs(val[:, 0] - (km + 4 * cos + kp) / 6.0).max() < 1e-14
    # and the analytic eigenvalue, to the fp32 rounding of the coefficients
    eig = (2.0 + np.cos(2 * np.pi * m / n)) / 3.0
    assert np.abs(val[:, 0] - np.cos(2 * np.pi * m * k / n) * eig).max() < 2e-7


# ----------------------------------------------------------------------------------------
# 6. lattice periodicity, including across the wrap seam, triclinic
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("lat", [TRICLINIC, SKEW])
def test_lattice_periodicity(lat):
    grid = (6, 5, 7)
    A, c, pos = workloads.small_case(grid, 4, 50, lat, seed=21, spread=1.0)
    v0, g0, l0, cell0 = oracle.eval_fast(A, grid, c, pos)
    for shift in [(1, 0, 0), (0, -1, 0), (0, 0, 1), (2, -3, 5)]:
        pos2 = pos + np.array(shift, dtype=np.float64) @ A
        v1, g1, l1, _ = oracle.eval_fast(A, grid, c, pos2)
        assert np.abs(v1 - v0).max() < 1e-11
        assert np.abs(g1 - g0).max() < 1e-10
        assert np.abs(l1 - l0).max() < 1e-9


# ----------------------------------------------------------------------------------------
# 7. gradient and Laplacian = central finite differences of the oracle's VALUES
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("lat,grid", [(ORTHO, (8, 8, 6)), (TRICLINIC, (7, 6, 8)), (SKEW, (5, 6, 7))])
def test_derivatives_by_finite_differences(lat, grid):
    A = np.array(lat, dtype=np.float64)
    rng = np.random.default_rng(33)
    c = rng.standard_normal((*grid, 3)).astype(np.float32)
    h = oracle.spacing(A, grid).min()
    # keep points away from knots (S''' jumps there): f in [0.2, 0.8]
    n = np.array(grid, dtype=np.float64)
    u = (rng.integers(0, grid, size=(40, 3)) + 0.2 + 0.6 * rng.random((40, 3))) / n
    pos = u @ A
    val, grad, lap, _ = oracle.eval_fast(A, grid, c, pos)
    d1 = 1e-5 * h
    scale = np.abs(grad).max()
    for x in range(3):
        e = np.zeros(3)
        e[x] = 1.0
        vp = oracle.eval_fast(A, grid, c, pos + d1 * e, mode=oracle.VALUE)[0]
        vm = oracle.eval_fast(A, grid, c, pos - d1 * e, mode=oracle.VALUE)[0]
        gfd = (vp - vm) / (2 * d1)
        assert np.abs(gfd - grad[:, x, :]).max() < 1e-8 * scale + 1e-9

    # Along a general Cartesian line the tricubic is a polynomial of degree up to 9, so the
    # second central difference carries an O(d^2) term: remove it by Richardson extrapolation.
    def second_difference(d):
        out = np.zeros_like(lap)
        for x in range(3):
            e = np.zeros(3)
            e[x] = 1.0
            vp = oracle.eval_fast(A, grid, c, pos + d * e, mode=oracle.VALUE)[0]
            vm = oracle.eval_fast(A, grid, c, pos - d * e, mode=oracle.VALUE)[0]
            out += (vp - 2 * val + vm) / (d * d)
        return out

    d2 = 4e-3 * h
    lap_fd = (4.0 * second_difference(d2 / 2) - second_difference(d2)) / 3.0
    assert np.abs(lap_fd - lap).max() < 1e-7 * np.abs(lap).max()


# ----------------------------------------------------------------------------------------
# 8. C2 continuity across cell faces (reading R10: either neighbour cell is "correct")
# ----------------------------------------------------------------------------------------
def test_continuity_across_cell_faces():
    grid = (6, 6, 6)
    A, c, _ = workloads.small_case(grid, 3, 1, SKEW, seed=5)
    n = np.array(grid, dtype=np.float64)
    rng = np.random.default_rng(9)
    eps = 1e-9
    for axis in range(3):
        u = rng.random((30, 3))
        u[:, axis] = rng.integers(0, grid[axis], size=30) / n[axis]
        um, up = u.copy(), u.copy()
        um[:, axis] -= eps / n[axis]
        up[:, axis] += eps / n[axis]
        vm, gm, lm, cm = oracle.eval_fast(A, grid, c, um @ A)
        vp, gp, lp, cp = oracle.eval_fast(A, grid, c, up @ A)
        assert np.any(cm[:, axis] != cp[:, axis])            # the face really was crossed
        assert np.abs(vm - vp).max() < 1e-7
        assert np.abs(gm - gp).max() < 1e-6
        assert np.abs(lm - lp).max() < 1e-5


# ----------------------------------------------------------------------------------------
# 9. separable special case -> library routine: scipy.interpolate.BSpline, uniform knots
# ----------------------------------------------------------------------------------------
def _scipy_periodic_1d(p, t, nu=0):
    """sum_k p[k mod n] B(t - k) with scipy: cubic BSpline on integer knots.  Basis j of
    knots -8..n+8 is supported on [j-8, j-4] and centred at j-6, so coefficient j = p[(j-6) % n]."""
    from scipy.interpolate import BSpline
    n = len(p)
    knots = np.arange(-8, n + 9, dtype=np.float64)
    nb = len(knots) - 4
    coef = np.array([p[(j - 6) % n] for j in range(nb)], dtype=np.float64)
    return BSpline(knots, coef, 3, extrapolate=False)(t, nu=nu)


def test_separable_coefficients_against_scipy_bspline():
    grid = (7, 6, 9)
    n = np.array(grid, dtype=np.float64)
    rng = np.random.default_rng(12)
    p, q, r = [rng.standard_normal(g).astype(np.float32) for g in grid]
    c = (p[:, None, None] * q[None, :, None] * r[None, None, :]).astype(np.float64)
    # the product must be exactly representable for an exact comparison: use fp32 products
    # re-rounded, and compare against scipy on the separately rounded 3-D table instead
    c32 = c.astype(np.float32)[..., None]
    lat = ((7.0, 0, 0), (0, 6.0, 0), (0, 0, 9.0))          # unit spacing, t = r
    u = rng.random((60, 3))
    pos = u * n
    val, grad, lap, _ = oracle.eval_fast(lat, grid, c32, pos)
    t = pos
    f = [_scipy_periodic_1d(v.astype(np.float64), t[:, a]) for a, v in enumerate((p, q, r))]
    f1 = [_scipy_periodic_1d(v.astype(np.float64), t[:, a], 1) for a, v in enumerate((p, q, r))]
    f2 = [_scipy_periodic_1d(v.astype(np.float64), t[:, a], 2) for a, v in enumerate((p, q, r))]
    tol = 5e-7 * np.abs(c).max()        # fp32 rounding of the product table
    assert np.abs(val[:, 0] - f[0] * f[1] * f[2]).max() < tol
    assert np.abs(grad[:, 0, 0] - f1[0] * f[1] * f[2]).max() < 4 * tol
    assert np.abs(grad[:, 1, 0] - f[0] * f1[1] * f[2]).max() < 4 * tol
    assert np.abs(grad[:, 2, 0] - f[0] * f[1] * f1[2]).max() < 4 * tol
    lap_ref = f2[0] * f[1] * f[2] + f[0] * f2[1] * f[2] + f[0] * f[1] * f2[2]
    assert np.abs(lap[:, 0] - lap_ref).max() < 16 * tol


def test_one_dimensional_profile_against_scipy_exactly():
    """coefficients varying along one axis only: no product rounding, so the comparison with
    scipy's BSpline (value, 1st, 2nd derivative) holds to fp64 rounding."""
    rng = np.random.default_rng(13)
    for axis, grid in enumerate([(9, 4, 5), (4, 8, 5), (5, 4, 10)]):
        n = grid[axis]
        p = rng.standard_normal(n).astype(np.float32)
        shape = [1, 1, 1]
        shape[axis] = n
        c = np.broadcast_to(p.reshape(shape), grid)[..., None].copy()
        lat = np.diag(np.array(grid, dtype=np.float64))
        pos = rng.random((80, 3)) * np.array(grid)
        val, grad, lap, _ = oracle.eval_fast(lat, grid, c, pos)
        t = pos[:, axis]
        assert np.abs(val[:, 0] - _scipy_periodic_1d(p.astype(np.float64), t)).max() < 1e-14
        assert np.abs(grad[:, axis, 0] - _scipy_periodic_1d(p.astype(np.float64), t, 1)).max() < 1e-13
        assert np.abs(lap[:, 0] - _scipy_periodic_1d(p.astype(np.float64), t, 2)).max() < 1e-12


# ----------------------------------------------------------------------------------------
# 10. the cell index map (pinned fp64 sequence)
# ----------------------------------------------------------------------------------------
def test_cell_index_exact_grid_planes_and_wrap():
    # tiny config: h = 10/16 = 0.625 is exact in binary, so r = k h sits exactly on a plane
    lat = ((10.0, 0, 0), (0, 10.0, 0), (0, 0, 10.0))
    grid = (16, 16, 16)
    ks = np.arange(-40, 41)
    pos = np.stack([ks * 0.625, ks * 0.625 + 0.3125, np.zeros_like(ks, dtype=float)], axis=1)
    cell, frac = oracle.cellmap(lat, grid, pos)
    assert np.array_equal(cell[:, 0], ks % 16)               # f = 0 belongs to the upper cell
    assert np.array_equal(frac[:, 0], np.zeros(len(ks)))
    assert np.array_equal(cell[:, 1], ks % 16)
    assert np.array_equal(frac[:, 1], np.full(len(ks), 0.5))
    assert np.all(cell[:, 2] == 0)


def test_cell_index_adversarial_inputs():
    lat = np.array(TRICLINIC)
    grid = (96, 96, 112)
    tiny = np.array([[-1e-300, -1e-300, -1e-300], [1e-300, 0.0, -0.0],
                     [-5e-324, 5e-324, -1e-17]])
    cell, frac = oracle.cellmap(lat, grid, tiny)
    assert cell.min() >= 0 and (cell < np.array(grid)).all()
    assert (frac >= 0).all() and (frac < 1).all()
    # u - floor(u) rounds to 1.0 for a tiny negative u: folded back to cell 0, f = 0
    assert np.array_equal(cell[0], [0, 0, 0]) and np.array_equal(frac[0], [0, 0, 0])
    # far away: +-1e3 cells, still in range and periodic with the home image to ~1e-10
    rng = np.random.default_rng(2)
    u = rng.random((500, 3))
    home, fh = oracle.cellmap(lat, grid, u @ lat)
    far, ff = oracle.cellmap(lat, grid, (u + np.array([1000, -1000, 777])) @ lat)
    assert far.min() >= 0 and (far < np.array(grid)).all()
    th, tf = home + fh, far + ff
    d = np.abs(th - tf)
    d = np.minimum(d, np.array(grid) - d)
    assert d.max() < 1e-8
    # 1 ulp either side of a plane
    x = 0.625 * 5
    lat2 = ((10.0, 0, 0), (0, 10.0, 0), (0, 0, 10.0))
    # either side of a plane (1 ulp below may legitimately round onto it: reading R10)
    pos = np.array([[x - 1e-12, 0, 0], [x, 0, 0], [np.nextafter(x, 10), 0, 0],
                    [np.nextafter(x, 0), 0, 0]])
    cell, frac = oracle.cellmap(lat2, (16, 16, 16), pos)
    assert list(cell[:3, 0]) == [4, 5, 5] and cell[3, 0] in (4, 5)
    assert frac[0, 0] < 1.0 and frac[1, 0] == 0.0


def test_cell_index_matches_exact_rational_arithmetic():
    """Away from cell faces the index is what exact arithmetic gives: checked with
    Python Fractions on a lattice with exactly representable entries."""
    lat = ((8.0, 0, 0), (2.0, 4.0, 0), (1.0, 0.5, 16.0))
    grid = (5, 7, 6)
    rng = np.random.default_rng(17)
    pos = (rng.integers(-2000, 2000, size=(200, 3)) / 64.0)          # dyadic rationals
    cell, frac = oracle.cellmap(lat, grid, pos)
    A = [[Fraction(x) for x in row] for row in lat]
    det = (A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1])
           - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0])
           + A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0]))
    # solve u A = r exactly by Cramer's rule on A^T
    def solve(r):
        At = [[A[j][i] for j in range(3)] for i in range(3)]          # At u = r
        out = []
        for col in range(3):
            Mx = [row[:] for row in At]
            for i in range(3):
                Mx[i][col] = r[i]
            d = (Mx[0][0] * (Mx[1][1] * Mx[2][2] - Mx[1][2] * Mx[2][1])
                 - Mx[0][1] * (Mx[1][0] * Mx[2][2] - Mx[1][2] * Mx[2][0])
                 + Mx[0][2] * (Mx[1][0] * Mx[2][1] - Mx[1][1] * Mx[2][0]))
            out.append(d / det)
        return out
    checked = 0
    for e in range(pos.shape[0]):
        u = solve([Fraction(float(x)) for x in pos[e]])
        for a in range(3):
            t = (u[a] - (u[a].numerator // u[a].denominator)) * grid[a]
            i_exact = t.numerator // t.denominator
            f_exact = float(t - i_exact)
            if min(f_exact, 1 - f_exact) < 1e-9:
                continue                                                 # on a face: R10
            assert cell[e, a] == i_exact
            assert abs(frac[e, a] - f_exact) < 1e-12
            checked += 1
    assert checked > 500


def test_non_finite_position_gives_nan_and_minus_one():
    A, c, pos = workloads.small_case((5, 5, 5), 2, 4, ORTHO, seed=1)
    pos[1, 2] = np.nan
    pos[3, 0] = np.inf
    val, grad, lap, cell = oracle.eval_fast(A, (5, 5, 5), c, pos)
    for e in (1, 3):
        assert np.isnan(val[e]).all() and np.isnan(grad[e]).all() and np.isnan(lap[e]).all()
        assert (cell[e] == -1).all()
    for e in (0, 2):
        assert np.isfinite(val[e]).all() and (cell[e] >= 0).all()


def test_spacing_values_of_the_five_configs():
    """h = max_a h_a of DESIGN.md reading R13, against hand arithmetic: orthorhombic h_a =
    L_a / n_a; triclinic h_a = V / (n_a |a_b x a_c|)."""
    for name, expect in [("tiny", 0.625), ("small", 0.25), ("tio2", 0.28)]:
        cfg = workloads.CONFIGS[name]
        assert abs(oracle.spacing(cfg.lattice, cfg.grid).max() - expect) < 1e-15
    cfg = workloads.CONFIGS["large"]
    A = np.array(cfg.lattice)
    V = abs(np.linalg.det(A))
    h = [V / (cfg.grid[a] * np.linalg.norm(np.cross(A[(a + 1) % 3], A[(a + 2) % 3])))
         for a in range(3)]
    assert np.abs(oracle.spacing(cfg.lattice, cfg.grid) - np.array(h)).max() < 1e-14
    assert abs(max(h) - 24.0 / 112.0) < 1e-15


# ------------------------------------------------------------------ contraction
def test_contract_one_hot_selects_an_orbital_and_constant_table_sums_d():
    """oracle.contract against what fixes it: d = e_k returns orbital k of eval_fast; a constant
    table c = kappa gives psi_l = kappa for every l (partition of unity), so out[0] = kappa sum(d)
    and the derivative entries vanish; linear in d."""
    rng = np.random.default_rng(5)
    A, c, pos = workloads.small_case((6, 5, 7), 9, 12, ((5.0, 0.3, -0.2), (1.1, 4.0, 0.7), (-0.6, 0.9, 6.0)), seed=3)
    val, grad, lap, _ = oracle.eval_fast(A, (6, 5, 7), c, pos)
    for k in (0, 4, 8):
        d = np.zeros((12, 9)); d[:, k] = 1.0
        out = oracle.contract(val, grad, lap, d)
        assert np.array_equal(out[:, 0], val[:, k]) and np.array_equal(out[:, 1:4], grad[:, :, k])
        assert np.array_equal(out[:, 4], lap[:, k])
    d1, d2 = rng.standard_normal((12, 9)), rng.standard_normal((12, 9))
    lhs = oracle.contract(val, grad, lap, 2.0 * d1 - 3.0 * d2)
    rhs = 2.0 * oracle.contract(val, grad, lap, d1) - 3.0 * oracle.contract(val, grad, lap, d2)
    assert np.allclose(lhs, rhs, rtol=0, atol=1e-10)
    kappa = np.full_like(c, 1.75)
    v2, g2, l2, _ = oracle.eval_fast(A, (6, 5, 7), kappa, pos)
    out = oracle.contract(v2, g2, l2, d1)
    assert np.allclose(out[:, 0], 1.75 * d1.sum(axis=1), rtol=0, atol=1e-12)
    assert np.abs(out[:, 1:]).max() < 1e-11
    vo = oracle.contract(val, None, None, d1)
    assert np.array_equal(vo[:, 0], oracle.contract(val, grad, lap, d1)[:, 0]) and not vo[:, 1:].any()


def test_contract_rows_equals_contract_and_its_pins():
    """oracle.contract_rows (numpy dot per position, used for full-size comparisons) against the
    loop form oracle.contract, and against the same one-hot / constant-table facts."""
    rng = np.random.default_rng(6)
    A, c, pos = workloads.small_case((6, 5, 7), 37, 40, ((5.0, 0.3, -0.2), (1.1, 4.0, 0.7), (-0.6, 0.9, 6.0)), seed=9)
    val, grad, lap, _ = oracle.eval_fast(A, (6, 5, 7), c, pos)
    d = rng.standard_normal((40, 37))
    a, b = oracle.contract(val, grad, lap, d), oracle.contract_rows(val, grad, lap, d)
    scale = np.abs(val).max() * np.abs(d).sum(axis=1).max()
    assert np.abs(a[:, 0] - b[:, 0]).max() <= 1e-14 * scale
    assert np.abs(a[:, 1:4] - b[:, 1:4]).max() <= 1e-14 * np.abs(grad).max() * np.abs(d).sum(axis=1).max()
    assert np.abs(a[:, 4] - b[:, 4]).max() <= 1e-14 * np.abs(lap).max() * np.abs(d).sum(axis=1).max()
    e = np.zeros((40, 37)); e[:, 11] = 1.0
    out = oracle.contract_rows(val, grad, lap, e)
    assert np.array_equal(out[:, 0], val[:, 11]) and np.array_equal(out[:, 1:4], grad[:, :, 11])
    assert np.array_equal(out[:, 4], lap[:, 11])
    vo = oracle.contract_rows(val, None, None, d)
    assert np.array_equal(vo[:, 0], b[:, 0]) and not vo[:, 1:].any()
