"""CPU fp64 oracle for the blip orbital evaluation (arxiv/paper_1204_1121, Eq. 6-8).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this.

`eval_fast`  — ctypes onto oracle/blip_oracle.c (the paper's algorithm, fp64, plain loops).
`blip_brute` — the definition summed over ALL grid sites (numpy, separate code).
"""
import ctypes
import numpy as np

from . import build as _build

VALUE, VGL = 0, 1
_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        fp = ctypes.POINTER(ctypes.c_float)
        L.blip_oracle_inverse_lattice.argtypes = [dp, dp]
        L.blip_oracle_inverse_lattice.restype = ctypes.c_int
        L.blip_oracle_cellmap.argtypes = [dp, ip, dp, ctypes.c_longlong, ip, dp]
        L.blip_oracle_cellmap.restype = ctypes.c_int
        L.blip_oracle_eval.argtypes = [dp, ip, ctypes.c_int, fp, dp, ctypes.c_longlong,
                                       ctypes.c_int, dp, dp, dp, ip]
        L.blip_oracle_eval.restype = ctypes.c_int
        L.blip_oracle_eval_hess.argtypes = [dp, ip, ctypes.c_int, fp, dp, ctypes.c_longlong, dp, dp, dp, ip]
        L.blip_oracle_eval_hess.restype = ctypes.c_int
        L.blip_oracle_spacing.argtypes = [dp, ip, dp]
        L.blip_oracle_spacing.restype = ctypes.c_int
        L.blip_oracle_num_threads.restype = ctypes.c_int
        L.blip_oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _i(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def _prep(lattice, grid):
    A = np.ascontiguousarray(np.asarray(lattice, dtype=np.float64).reshape(9))
    n = np.ascontiguousarray(np.asarray(grid, dtype=np.int32).reshape(3))
    return A, n


def inverse_lattice(lattice):
    A = np.ascontiguousarray(np.asarray(lattice, dtype=np.float64).reshape(9))
    G = np.empty(9, dtype=np.float64)
    if lib().blip_oracle_inverse_lattice(_d(A), _d(G)):
        raise ValueError("singular or non-finite lattice")
    return G.reshape(3, 3)


def cellmap(lattice, grid, positions):
    A, n = _prep(lattice, grid)
    pos = np.ascontiguousarray(np.asarray(positions, dtype=np.float64).reshape(-1, 3))
    M = pos.shape[0]
    cell = np.empty((M, 3), dtype=np.int32)
    frac = np.empty((M, 3), dtype=np.float64)
    if lib().blip_oracle_cellmap(_d(A), _i(n), _d(pos), M, _i(cell), _d(frac)):
        raise ValueError("singular or non-finite lattice")
    return cell, frac


def eval_fast(lattice, grid, coeffs, positions, mode=VGL):
    """Returns (val [M][L], grad [M][3][L] or None, lap [M][L] or None, cell [M][3]) in fp64."""
    A, n = _prep(lattice, grid)
    c = np.ascontiguousarray(coeffs, dtype=np.float32)
    assert c.ndim == 4 and tuple(c.shape[:3]) == tuple(int(x) for x in n), c.shape
    L = c.shape[3]
    pos = np.ascontiguousarray(np.asarray(positions, dtype=np.float64).reshape(-1, 3))
    M = pos.shape[0]
    val = np.empty((M, L), dtype=np.float64)
    cell = np.empty((M, 3), dtype=np.int32)
    if mode == VGL:
        grad = np.empty((M, 3, L), dtype=np.float64)
        lap = np.empty((M, L), dtype=np.float64)
        gp, lp = _d(grad), _d(lap)
    else:
        grad = lap = None
        gp = lp = ctypes.POINTER(ctypes.c_double)()
    rc = lib().blip_oracle_eval(_d(A), _i(n), L,
                                c.ctypes.data_as(ctypes.POINTER(ctypes.c_float)),
                                _d(pos), M, mode, _d(val), gp, lp, _i(cell))
    if rc:
        raise ValueError(f"blip_oracle_eval failed with code {rc}")
    return val, grad, lap, cell


HESS_COMPONENTS = ((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2))     # xx yy zz xy xz yz


def eval_hess(lattice, grid, coeffs, positions):
    """Value, Cartesian gradient and full Cartesian Hessian (blip_oracle_eval_hess): returns
    (val [M][L], grad [M][3][L], hess [M][6][L] in the order xx yy zz xy xz yz, cell [M][3]), fp64."""
    A, n = _prep(lattice, grid)
    c = np.ascontiguousarray(coeffs, dtype=np.float32)
    assert c.ndim == 4 and tuple(c.shape[:3]) == tuple(int(x) for x in n), c.shape
    L = c.shape[3]
    pos = np.ascontiguousarray(np.asarray(positions, dtype=np.float64).reshape(-1, 3))
    M = pos.shape[0]
    val = np.empty((M, L), dtype=np.float64)
    grad = np.empty((M, 3, L), dtype=np.float64)
    hess = np.empty((M, 6, L), dtype=np.float64)
    cell = np.empty((M, 3), dtype=np.int32)
    rc = lib().blip_oracle_eval_hess(_d(A), _i(n), L, c.ctypes.data_as(ctypes.POINTER(ctypes.c_float)),
                                     _d(pos), M, _d(val), _d(grad), _d(hess), _i(cell))
    if rc:
        raise ValueError(f"blip_oracle_eval_hess failed with code {rc}")
    return val, grad, hess, cell


def bloch(val, grad, lap, kpoints, positions):
    """Complex orbitals with a per-orbital Bloch phase (the paper's orbitals
    are complex, "2 components in complex numbers").  Complex orbital m is made of the
    real channels (2m, 2m+1) of the table — u_m = S_{2m} + i S_{2m+1}, periodic in the cell — times
    the phase of its k-point [DESIGN.md reading R8a; the paper does not write the phase out]:

        psi_m(r)       = exp(i k_m . r) u_m(r)
        grad psi_m     = exp(i k_m . r) (grad u_m + i k_m u_m)                          (product rule)
        laplace psi_m  = exp(i k_m . r) (laplace u_m + 2 i k_m . grad u_m - |k_m|^2 u_m)

    val [M][L], grad [M][3][L], lap [M][L]: oracle results (fp64) for the real channels, L even;
    kpoints [L/2][3] Cartesian (rad / bohr); positions [M][3] Cartesian.  grad / lap may be None.
    Returns complex128 (psi [M][L/2], gpsi [M][3][L/2] or None, lpsi [M][L/2] or None).
    Pins (tests/test_oracle_pins.py): k = 0 returns the real channels; |psi|^2 does not depend on k;
    a constant table gives a plane wave (grad = i k psi, laplace = -|k|^2 psi); central differences
    of psi VALUES; psi(r + a_j) = exp(i k . a_j) psi(r)."""
    val = np.asarray(val, dtype=np.float64)
    k = np.asarray(kpoints, dtype=np.float64).reshape(-1, 3)
    r = np.asarray(positions, dtype=np.float64).reshape(-1, 3)
    M, L = val.shape
    assert L % 2 == 0 and k.shape[0] == L // 2 and r.shape[0] == M
    Lc = L // 2
    psi = np.empty((M, Lc), dtype=np.complex128)
    gpsi = None if grad is None else np.empty((M, 3, Lc), dtype=np.complex128)
    lpsi = None if lap is None else np.empty((M, Lc), dtype=np.complex128)
    for m in range(Lc):
        theta = r[:, 0] * k[m, 0] + r[:, 1] * k[m, 1] + r[:, 2] * k[m, 2]
        phase = np.cos(theta) + 1j * np.sin(theta)
        u = val[:, 2 * m] + 1j * val[:, 2 * m + 1]
        psi[:, m] = phase * u
        if grad is not None:
            gu = grad[:, :, 2 * m] + 1j * grad[:, :, 2 * m + 1]                 # [M][3]
            gpsi[:, :, m] = phase[:, None] * (gu + 1j * k[m][None, :] * u[:, None])
            if lap is not None:
                lu = lap[:, 2 * m] + 1j * lap[:, 2 * m + 1]
                kg = gu[:, 0] * k[m, 0] + gu[:, 1] * k[m, 1] + gu[:, 2] * k[m, 2]
                lpsi[:, m] = phase * (lu + 2j * kg - (k[m] @ k[m]) * u)
    return psi, gpsi, lpsi


def spacing(lattice, grid):
    """Perpendicular grid-plane spacings h_a (reading R13)."""
    A, n = _prep(lattice, grid)
    h = np.empty(3, dtype=np.float64)
    if lib().blip_oracle_spacing(_d(A), _i(n), _d(h)):
        raise ValueError("singular or non-finite lattice")
    return h


def num_threads():
    return int(lib().blip_oracle_num_threads())


def set_num_threads(t):
    lib().blip_oracle_set_num_threads(int(t))


def contract(val, grad, lap, d):
    """Orbital-axis contraction of oracle results with per-position vectors d [M][L]
    (Eq. 11, 395-399 §VI.D: sum_l psi_l(r'_j) (D^-1)_lj), written out as the
    definition, one position and one orbital at a time in fp64:
        out[j] = (sum_l val[j][l] d[j][l],  sum_l grad[j][i][l] d[j][l] (i = x, y, z),  sum_l lap[j][l] d[j][l])
    grad / lap may be None (value only: entries 1..4 stay zero).
    Pins (tests/test_oracle_pins.py): a one-hot d selects one orbital; a constant table gives the sum of d."""
    val = np.asarray(val, dtype=np.float64)
    d = np.asarray(d, dtype=np.float64)
    M, L = val.shape
    out = np.zeros((M, 5), dtype=np.float64)
    for j in range(M):
        s = np.zeros(5)
        for l in range(L):
            w = d[j, l]
            s[0] += val[j, l] * w
            if grad is not None:
                s[1] += grad[j, 0, l] * w
                s[2] += grad[j, 1, l] * w
                s[3] += grad[j, 2, l] * w
                s[4] += lap[j, l] * w
        out[j] = s
    return out


def contract_rows(val, grad, lap, d):
    """The same contraction as `contract`, one position at a time with numpy's fp64 dot product as
    the library primitive for the sum over l (Eq. 11: sum_l psi_l(r'_j) (D^-1)_lj).
    For full-size comparisons, where the pure-Python double loop of `contract` would take minutes.
    Pin (tests/test_oracle_pins.py): equal to `contract` on a seeded case to fp64 rounding, and the
    one-hot / constant-table pins of `contract`."""
    val = np.asarray(val, dtype=np.float64)
    d = np.asarray(d, dtype=np.float64)
    M = val.shape[0]
    out = np.zeros((M, 5), dtype=np.float64)
    for j in range(M):
        out[j, 0] = np.dot(val[j], d[j])
        if grad is not None:
            out[j, 1] = np.dot(grad[j, 0], d[j])
            out[j, 2] = np.dot(grad[j, 1], d[j])
            out[j, 3] = np.dot(grad[j, 2], d[j])
            out[j, 4] = np.dot(lap[j], d[j])
    return out
