"""Complex orbitals with a per-orbital Bloch phase (blipgpu_set_kpoints / blipgpu_eval_complex;
SURVEY.md §8f NEXT-4) against oracle.bloch applied to the oracle's real channels.

Tolerance (reading R8a): psi = e^{i theta}(u_re + i u_im), so each of Re psi, Im psi
mixes the errors of both channels — |cos| + |sin| <= sqrt 2, taken as 2 to also cover the phase
rounding (k.r is reduced in fp64; what is left is the fp32 rounding of an angle in (-pi, pi],
< 2e-7 rad, against a relative tolerance of 2e-5):
    value     2 tol_val
    gradient  2 (tol_grad + |k| tol_val)                                 (grad u + i k u)
    Laplacian 2 (tol_lap + 2 sqrt3 |k| tol_grad + |k|^2 tol_val)          (lap u + 2 i k.grad u - k^2 u)
with tol_* north_star's tolerances of the real channels and |k| the largest k-point norm."""
import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import tolerances, torch_cuda, blip  # noqa: F401 (fixtures)

pytestmark = pytest.mark.gpu

TRICLINIC = ((20.0, 0.0, 0.0), (3.0, 19.0, 0.0), (2.0, 2.0, 24.0))
ORTHO = ((7.0, 0.0, 0.0), (0.0, 8.5, 0.0), (0.0, 0.0, 9.25))


def run_complex(torch, blip, t, pos, L, mode=1, ld=None):
    M = pos.shape[0]
    ld = (L + 3) // 4 * 4 if ld is None else ld
    val = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda")
    grad = torch.full((M, 3, ld), 7.0, dtype=torch.float32, device="cuda") if mode else None
    lap = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda") if mode else None
    cell = torch.empty((M, 3), dtype=torch.int32, device="cuda")
    blip.blipgpu_eval_complex(t.handle, torch.from_numpy(np.ascontiguousarray(pos)).cuda(), M, mode, val, grad, lap, ld, cell)
    torch.cuda.synchronize()

    def cplx(x):
        if x is None:
            return None
        x = x.cpu().numpy()[..., :L].astype(np.float64)
        return x[..., 0::2] + 1j * x[..., 1::2]

    return cplx(val), cplx(grad), cplx(lap), cell.cpu().numpy()


def complex_tolerances(A, grid, cmax, k):
    tv, tg, tl = tolerances(A, grid, cmax)
    kmax = float(np.linalg.norm(k, axis=1).max())
    return 2 * tv, 2 * (tg + kmax * tv), 2 * (tl + 2 * np.sqrt(3.0) * kmax * tg + kmax ** 2 * tv)


def check(A, grid, c, pos, k, out, mode=1):
    oval, ograd, olap, ocell = oracle.eval_fast(A, grid, c, pos, mode=mode)
    psi, gpsi, lpsi = oracle.bloch(oval, ograd, olap, k, pos)
    tv, tg, tl = complex_tolerances(A, grid, float(np.abs(c).max()), k)
    assert np.array_equal(out[3], ocell)

    def err(a, b):
        d = a - b
        return max(float(np.abs(d.real).max()), float(np.abs(d.imag).max()))

    assert err(out[0], psi) <= tv
    if mode:
        assert err(out[1], gpsi) <= tg
        assert err(out[2], lpsi) <= tl
        return err(out[0], psi) / tv, err(out[1], gpsi) / tg, err(out[2], lpsi) / tl


@pytest.mark.parametrize("grid,L,M,lat,path", [
    ((9, 10, 13), 130, 3000, TRICLINIC, 2),                 # staged kernel, ragged orbital tile
    ((9, 10, 13), 130, 3000, TRICLINIC, 1),                 # direct kernel, grouped
    ((6, 5, 7), 38, 300, TRICLINIC, 0),                     # split kernel
    ((11, 9, 14), 140, 5000, ORTHO, 2),                     # diagonal-lattice mode of the kernels
    ((11, 9, 14), 258, 2500, ORTHO, 1),
])
def test_complex_small_cases(torch_cuda, blip, grid, L, M, lat, path):
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=L + M, spread=6.0)        # |k.r| up to a few tens of radians
    k = workloads.kpoints(A, L // 2, seed=L)
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_kpoints(t.handle, k)
    blip.blipgpu_set_tuning(t.handle, path=path)
    for mode in (1, 0):
        out = run_complex(torch_cuda, blip, t, pos, L, mode=mode, ld=(L + 3) // 4 * 4 + 4)
        assert blip.blipgpu_last_path(t.handle) == (path if path else 3)
        check(A, grid, c, pos, k, out, mode=mode)
    t.close()


def test_complex_zero_k_returns_the_bits_of_the_real_path(torch_cuda, blip):
    torch = torch_cuda
    grid, L, M = (9, 10, 13), 130, 3000
    A, c, pos = workloads.small_case(grid, L, M, TRICLINIC, seed=4, spread=3.0)
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_kpoints(t.handle, np.zeros((L // 2, 3)))
    dpos = torch.from_numpy(pos).cuda()
    for path in (2, 1):
        blip.blipgpu_set_tuning(t.handle, path=path)
        real = t.eval(dpos, mode=blip.VGL)
        ld = t.ld
        val = torch.empty((M, ld), dtype=torch.float32, device="cuda")
        grad = torch.empty((M, 3, ld), dtype=torch.float32, device="cuda")
        lap = torch.empty((M, ld), dtype=torch.float32, device="cuda")
        blip.blipgpu_eval_complex(t.handle, dpos, M, blip.VGL, val, grad, lap, ld)
        torch.cuda.synchronize()
        assert torch.equal(val[:, :L], real[0]) and torch.equal(grad[:, :, :L], real[1]) and torch.equal(lap[:, :L], real[2])
    t.close()


def test_complex_far_positions_non_finite_and_errors(torch_cuda, blip):
    """Positions hundreds of cells away (|k.r| ~ 1e3 rad: the phase must not lose accuracy), a
    non-finite position, and the argument errors of the two calls."""
    grid, L = (8, 8, 8), 12
    A, c, pos = workloads.small_case(grid, L, 64, TRICLINIC, seed=1, spread=400.0)
    k = workloads.kpoints(A, L // 2, seed=7)
    pos[7, 2] = np.nan
    t = blip.BlipTable(A, grid, L, c)
    lib = blip.lib()
    dummy = torch_cuda.empty((64, 12), dtype=torch_cuda.float32, device="cuda")
    q = lambda x: x.data_ptr()
    assert lib.blipgpu_eval_complex(t.handle, q(dummy), 1, 0, q(dummy), None, None, 12, None, None) == blip.EINVAL   # no k-points yet
    blip.blipgpu_set_kpoints(t.handle, k)
    out = run_complex(torch_cuda, blip, t, pos, L)
    assert np.isnan(out[0][7]).all() and np.isnan(out[1][7]).all() and np.isnan(out[2][7]).all()
    good = np.arange(64) != 7
    check(A, grid, c, pos[good], k, tuple(x[good] for x in out))
    assert lib.blipgpu_eval_complex(t.handle, q(dummy), 1, blip.VGH, q(dummy), q(dummy), q(dummy), 12, None, None) == blip.EINVAL
    bad = k.copy(); bad[0, 0] = np.inf
    assert lib.blipgpu_set_kpoints(t.handle, bad.ctypes.data) == blip.EINVAL
    blip.blipgpu_set_kpoints(t.handle, None)
    assert lib.blipgpu_eval_complex(t.handle, q(dummy), 1, 0, q(dummy), None, None, 12, None, None) == blip.EINVAL
    t.close()
    A, c, pos = workloads.small_case((6, 6, 6), 7, 4, TRICLINIC, seed=1)
    t = blip.BlipTable(A, (6, 6, 6), 7, c)                                          # odd number of real channels
    assert lib.blipgpu_set_kpoints(t.handle, np.zeros((3, 3)).ctypes.data) == blip.EINVAL
    t.close()


def test_complex_tio2_full_size_every_output(torch_cuda, blip):
    """The bench configuration as the paper's workload has it: 384 complex orbitals (768 real
    channels), 49,152 positions, staged kernel; every output against the oracle."""
    cfg = workloads.CONFIGS["tio2"]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    pos = workloads.positions(cfg)
    k = workloads.kpoints(A, cfg.norb // 2)
    t = blip.BlipTable(A, cfg.grid, cfg.norb, c)
    blip.blipgpu_set_kpoints(t.handle, k)
    out = run_complex(torch_cuda, blip, t, pos, cfg.norb)
    assert blip.blipgpu_last_path(t.handle) == 2
    t.close()
    worst = (0, 0, 0)
    for lo in range(0, pos.shape[0], 8192):
        sl = slice(lo, min(lo + 8192, pos.shape[0]))
        w = check(A, cfg.grid, c, pos[sl], k, tuple(x[sl] for x in out))
        worst = tuple(max(a, b) for a, b in zip(worst, w))
    assert max(worst) < 0.5, worst
