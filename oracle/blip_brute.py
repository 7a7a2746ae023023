"""Brute-force DEFINITION of the blip expansion, summed over ALL grid sites (numpy, fp64).

TEST INFRASTRUCTURE ONLY.  Used to pin oracle/blip_oracle.c on tiny grids; shares nothing
with it (no cell search, no weight polynomials, library matrix inverse instead of the
pinned cofactor sequence).

Definition (the plain form of PAPER.md:78-86 Eq. 6-7 before the 64-site
restriction of PAPER.md:82 drops the exact zeros):

    S_l(r) = sum over every grid site k = (k1,k2,k3) of c[k][l] * prod_a Bper_a(t_a - k_a),
    t = n * (r . A^-1),   Bper_a(x) = sum over integer images m of B(x + m n_a),

B the centred cardinal cubic B-spline [not printed in the paper; textbook]:

    B(x) = 2/3 - x^2 + |x|^3/2      for |x| <= 1
           (2 - |x|)^3 / 6          for 1 <= |x| < 2
           0                        otherwise.

Gradient and Laplacian are the Cartesian derivatives of S_l, from the analytic B', B''.
"""
import numpy as np


def B(x):
    ax = np.abs(x)
    return np.where(ax <= 1.0, 2.0 / 3.0 - ax ** 2 + 0.5 * ax ** 3,
                    np.where(ax < 2.0, (2.0 - ax) ** 3 / 6.0, 0.0))


def dB(x):
    ax = np.abs(x)
    sg = np.sign(x)
    return np.where(ax <= 1.0, -2.0 * x + 1.5 * x * ax,
                    np.where(ax < 2.0, -sg * 0.5 * (2.0 - ax) ** 2, 0.0))


def d2B(x):
    ax = np.abs(x)
    return np.where(ax <= 1.0, -2.0 + 3.0 * ax, np.where(ax < 2.0, 2.0 - ax, 0.0))


def _periodic(fn, t, n, images):
    """fn summed over periodic images: out[k] = sum_m fn(t - k + m n), k = 0..n-1."""
    k = np.arange(n, dtype=np.float64)
    x = t - k
    # the nearest image of each site, then `images` more on either side
    m0 = np.round(-x / n)
    out = np.zeros(n, dtype=np.float64)
    for dm in range(-images, images + 1):
        out += fn(x + (m0 + dm) * n)
    return out


def eval_brute(lattice, grid, coeffs, positions, images=2, want_hessian=False):
    """Returns (val [M][L], grad [M][3][L], lap [M][L]) in fp64 — sum over all n1*n2*n3 sites;
    with want_hessian also the Cartesian Hessian [M][3][3][L] as a fourth entry."""
    A = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
    n = [int(x) for x in grid]
    c = np.asarray(coeffs, dtype=np.float64)
    assert c.shape[:3] == tuple(n)
    L = c.shape[3]
    pos = np.asarray(positions, dtype=np.float64).reshape(-1, 3)
    M = pos.shape[0]
    Ainv = np.linalg.inv(A)                       # u = r @ Ainv
    # dt_a/dr_i = n_a * Ainv[i][a]
    Jm = np.array([[n[a] * Ainv[i, a] for i in range(3)] for a in range(3)])
    val = np.zeros((M, L))
    grad = np.zeros((M, 3, L))
    lap = np.zeros((M, L))
    hess = np.zeros((M, 3, 3, L))
    for e in range(M):
        t = (pos[e] @ Ainv) * np.array(n, dtype=np.float64)
        b = [_periodic(B, t[a], n[a], images) for a in range(3)]
        b1 = [_periodic(dB, t[a], n[a], images) for a in range(3)]
        b2 = [_periodic(d2B, t[a], n[a], images) for a in range(3)]

        def contract(x, y, z):
            return np.einsum("i,j,k,ijkl->l", x, y, z, c)

        val[e] = contract(b[0], b[1], b[2])
        dt = np.stack([contract(b1[0], b[1], b[2]),
                       contract(b[0], b1[1], b[2]),
                       contract(b[0], b[1], b1[2])])          # [3][L]  dS/dt_a
        Ht = np.zeros((3, 3, L))                              # d2S/dt_a dt_b
        Ht[0, 0] = contract(b2[0], b[1], b[2])
        Ht[1, 1] = contract(b[0], b2[1], b[2])
        Ht[2, 2] = contract(b[0], b[1], b2[2])
        Ht[0, 1] = Ht[1, 0] = contract(b1[0], b1[1], b[2])
        Ht[0, 2] = Ht[2, 0] = contract(b1[0], b[1], b1[2])
        Ht[1, 2] = Ht[2, 1] = contract(b[0], b1[1], b1[2])
        grad[e] = Jm.T @ dt                                   # grad_i = sum_a J[a][i] dS/dt_a
        Hc = np.einsum("ai,abl,bj->ijl", Jm, Ht, Jm)          # Cartesian Hessian
        lap[e] = Hc[0, 0] + Hc[1, 1] + Hc[2, 2]
        hess[e] = Hc
    if want_hessian:
        return val, grad, lap, hess
    return val, grad, lap
