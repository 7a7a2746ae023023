"""blipgpu_eval_f64 (fp64 weights, accumulation and outputs from the resident
fp32 table) against the CPU fp64 oracle.  Both sides work in fp64 on the same fp32
coefficients widened exactly, so they differ by summation order only: tolerance 1e-12 x the
scale of each quantity (max|c|, max|c|/h, max|c|/h^2) — seven orders of magnitude tighter than
the fp32 path's, which makes this the sharpest check of indexing, weights and metric on the GPU."""
import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import torch_cuda, blip  # noqa: F401 (fixtures)

pytestmark = pytest.mark.gpu

TRICLINIC = ((20.0, 0.0, 0.0), (3.0, 19.0, 0.0), (2.0, 2.0, 24.0))
SKEW = ((5.0, 0.3, -0.2), (1.1, 4.0, 0.7), (-0.6, 0.9, 6.0))


def run_f64(torch, blip, t, pos, L, mode=1, ld=None):
    M = pos.shape[0]
    ld = (L + 3) // 4 * 4 if ld is None else ld
    val = torch.full((M, ld), 7.0, dtype=torch.float64, device="cuda")
    grad = torch.full((M, 3, ld), 7.0, dtype=torch.float64, device="cuda") if mode else None
    lap = torch.full((M, ld), 7.0, dtype=torch.float64, device="cuda") if mode else None
    cell = torch.empty((M, 3), dtype=torch.int32, device="cuda")
    blip.blipgpu_eval_f64(t.handle, torch.from_numpy(np.ascontiguousarray(pos)).cuda(), M, mode, val, grad, lap, ld, cell)
    torch.cuda.synchronize()
    assert blip.blipgpu_last_path(t.handle) == 4
    return (val.cpu().numpy()[:, :L], None if grad is None else grad.cpu().numpy()[:, :, :L],
            None if lap is None else lap.cpu().numpy()[:, :L], cell.cpu().numpy())


def check(A, grid, c, pos, out, mode=1):
    oval, ograd, olap, ocell = oracle.eval_fast(A, grid, c, pos, mode=mode)
    cmax = float(np.abs(c).max())
    h = float(oracle.spacing(A, grid).min())
    assert np.array_equal(out[3], ocell)
    assert np.abs(out[0] - oval).max() <= 1e-12 * cmax
    if mode:
        assert np.abs(out[1] - ograd).max() <= 1e-12 * cmax / h
        assert np.abs(out[2] - olap).max() <= 1e-12 * cmax / (h * h)


@pytest.mark.parametrize("grid,L,M,lat", [((6, 5, 7), 37, 300, SKEW), ((9, 10, 13), 130, 2000, TRICLINIC),
                                          ((4, 4, 4), 5, 100, SKEW), ((16, 16, 16), 32, 64, ((10.0, 0, 0), (0, 10.0, 0), (0, 0, 10.0)))])
def test_f64_small_cases(torch_cuda, blip, grid, L, M, lat):
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=L + M, spread=4.0)
    t = blip.BlipTable(A, grid, L, c)
    for mode in (1, 0):
        check(A, grid, c, pos, run_f64(torch_cuda, blip, t, pos, L, mode=mode, ld=(L + 3) // 4 * 4 + 4), mode=mode)
    t.close()


def test_f64_non_finite_and_errors(torch_cuda, blip):
    A, c, pos = workloads.small_case((8, 8, 8), 12, 40, TRICLINIC, seed=2)
    pos[3, 0] = np.inf
    t = blip.BlipTable(A, (8, 8, 8), 12, c)
    val, grad, lap, cell = run_f64(torch_cuda, blip, t, pos, 12)
    assert np.isnan(val[3]).all() and np.isnan(grad[3]).all() and np.isnan(lap[3]).all() and (cell[3] == -1).all()
    good = np.arange(40) != 3
    check(A, (8, 8, 8), c, pos[good], (val[good], grad[good], lap[good], cell[good]))
    L = blip.lib()
    assert L.blipgpu_eval_f64(t.handle, None, 4, 1, None, None, None, 12, None, None) == blip.EINVAL
    assert L.blipgpu_eval_f64(t.handle, None, 0, 1, None, None, None, 12, None, None) == blip.OK
    assert L.blipgpu_eval_f64(t.handle, None, 4, 1, None, None, None, 10, None, None) == blip.EINVAL
    t.close()


def test_f64_tio2_sampled_and_fp32_path_against_it(torch_cuda, blip):
    """1,536 positions of the TiO2 configuration: the fp64 kernel against the oracle, and the fp32
    staged/split results of the same positions against the fp64 kernel within north_star's tolerances."""
    torch = torch_cuda
    cfg = workloads.CONFIGS["tio2"]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    pos = workloads.positions(cfg, M=1536)
    t = blip.BlipTable(A, cfg.grid, cfg.norb, c)
    out = run_f64(torch, blip, t, pos, cfg.norb)
    check(A, cfg.grid, c, pos, out)
    val, grad, lap, cell = t.eval(torch.from_numpy(pos).cuda(), mode=blip.VGL, want_cell=True)
    cmax = float(np.abs(c).max())
    h = float(oracle.spacing(A, cfg.grid).max())
    assert np.abs(val.cpu().numpy() - out[0]).max() <= 2e-5 * cmax
    assert np.abs(grad.cpu().numpy() - out[1]).max() <= 2e-5 * cmax / h
    assert np.abs(lap.cpu().numpy() - out[2]).max() <= 5e-5 * cmax / h ** 2
    t.close()


def test_f64_tio2_full_size_every_output(torch_cuda, blip):
    """All 49,152 positions x 768 orbitals of the TiO2 configuration through blipgpu_eval_f64, every
    output against the oracle at the fp64 tolerance, in slabs of 8,192 positions (the fp64 outputs
    of the whole batch would be 1.5 GB on each side)."""
    cfg = workloads.CONFIGS["tio2"]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    pos = workloads.positions(cfg)
    t = blip.BlipTable(A, cfg.grid, cfg.norb, c)
    try:
        for lo in range(0, pos.shape[0], 8192):
            p = pos[lo:lo + 8192]
            check(A, cfg.grid, c, p, run_f64(torch_cuda, blip, t, p, cfg.norb))
    finally:
        t.close()


def test_f64_meets_the_bound_on_strongly_anisotropic_grids(torch_cuda, blip):
    """DESIGN.md reading R13a: beyond a spacing ratio of ~10 the fp32 kernels' Laplacian rounding
    (which scales with 1 / h_min^2) can pass north_star's bound (stated with h_max);
    blipgpu_eval_f64 is what such tables are given.  Grid 8 x 8 x 32 on a 4.3 x 11.4 x 3.6 cell
    (ratio 12.7) and a harsher 6 x 40 x 6 on 9 x 1.5 x 9 (ratio 40): the fp64 path meets north_star's
    fp32 bound with h = h_max by orders of magnitude, and its own 1e-12 bound with h_min."""
    for grid, lat, L, M in (((8, 8, 32), np.diag([4.3, 11.4, 3.6]), 130, 3000), ((6, 40, 6), np.diag([9.0, 1.5, 9.0]), 24, 500)):
        A, c, pos = workloads.small_case(grid, L, M, lat, seed=sum(grid))
        sp = oracle.spacing(A, grid)
        assert sp.max() / sp.min() > 12
        t = blip.BlipTable(A, grid, L, c)
        try:
            out = run_f64(torch_cuda, blip, t, pos, L)
            check(A, grid, c, pos, out)                       # 1e-12 with h_min
            oval, ograd, olap, _ = oracle.eval_fast(A, grid, c, pos)
            cmax, h = float(np.abs(c).max()), float(sp.max())
            assert np.abs(out[0] - oval).max() <= 1e-6 * 2e-5 * cmax
            assert np.abs(out[1] - ograd).max() <= 1e-6 * 2e-5 * cmax / h
            assert np.abs(out[2] - olap).max() <= 1e-4 * 5e-5 * cmax / h ** 2
        finally:
            t.close()
