"""Full Cartesian Hessian output (mode BLIPGPU_VGH) of
blipgpu_eval (fp32), blipgpu_eval_host and blipgpu_eval_f64 against oracle.eval_hess.

Tolerances: fp32 — every Hessian component within north_star's Laplacian tolerance
5e-5 max|c| / h^2 (a component is a sum of the same second-derivative terms the Laplacian adds up),
value and gradient within theirs; fp64 — 1e-12 x the scale of each quantity (summation order only)."""
import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import tolerances, torch_cuda, blip  # noqa: F401 (fixtures)

pytestmark = pytest.mark.gpu

TRICLINIC = ((20.0, 0.0, 0.0), (3.0, 19.0, 0.0), (2.0, 2.0, 24.0))
SKEW = ((5.0, 0.3, -0.2), (1.1, 4.0, 0.7), (-0.6, 0.9, 6.0))
ORTHO = ((7.0, 0.0, 0.0), (0.0, 8.5, 0.0), (0.0, 0.0, 9.25))


def run_vgh(torch, blip, t, pos, L, dtype, ld=None):
    M = pos.shape[0]
    ld = (L + 3) // 4 * 4 if ld is None else ld
    tt = torch.float32 if dtype == "f32" else torch.float64
    val = torch.full((M, ld), 7.0, dtype=tt, device="cuda")
    grad = torch.full((M, 3, ld), 7.0, dtype=tt, device="cuda")
    hess = torch.full((M, 6, ld), 7.0, dtype=tt, device="cuda")
    cell = torch.empty((M, 3), dtype=torch.int32, device="cuda")
    dpos = torch.from_numpy(np.ascontiguousarray(pos)).cuda()
    fn = blip.blipgpu_eval if dtype == "f32" else blip.blipgpu_eval_f64
    fn(t.handle, dpos, M, blip.VGH, val, grad, hess, ld, cell)
    torch.cuda.synchronize()
    assert blip.blipgpu_last_path(t.handle) == 4
    return val.cpu().numpy()[:, :L], grad.cpu().numpy()[:, :, :L], hess.cpu().numpy()[:, :, :L], cell.cpu().numpy()


def check(A, grid, c, pos, out, dtype):
    oval, ograd, ohess, ocell = oracle.eval_hess(A, grid, c, pos)
    cmax = float(np.abs(c).max())
    assert np.array_equal(out[3], ocell)
    if dtype == "f32":
        tv, tg, tl = tolerances(A, grid, cmax)
    else:
        h = float(oracle.spacing(A, grid).min())
        tv, tg, tl = 1e-12 * cmax, 1e-12 * cmax / h, 1e-12 * cmax / (h * h)
    assert np.abs(out[0] - oval).max() <= tv
    assert np.abs(out[1] - ograd).max() <= tg
    err = np.abs(out[2] - ohess).max(axis=(0, 2))            # per component
    assert (err <= tl).all(), err / tl
    return err / tl


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("grid,L,M,lat", [((6, 5, 7), 37, 300, SKEW), ((9, 10, 13), 130, 2500, TRICLINIC),
                                          ((4, 4, 4), 5, 100, SKEW), ((11, 9, 14), 140, 600, ORTHO)])
def test_hessian_small_cases(torch_cuda, blip, dtype, grid, L, M, lat):
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=L + M, spread=4.0)
    t = blip.BlipTable(A, grid, L, c)
    check(A, grid, c, pos, run_vgh(torch_cuda, blip, t, pos, L, dtype, ld=(L + 3) // 4 * 4 + 4), dtype)
    t.close()


def test_hessian_trace_matches_the_vgl_laplacian_and_table_eval(torch_cuda, blip):
    """BlipTable.eval(mode=VGH); the trace of the fp32 Hessian against the Laplacian the fast
    kernels return for the same positions (two tolerances apart at most)."""
    torch = torch_cuda
    grid, L, M = (9, 10, 13), 130, 3000
    A, c, pos = workloads.small_case(grid, L, M, TRICLINIC, seed=3, spread=3.0)
    t = blip.BlipTable(A, grid, L, c)
    dpos = torch.from_numpy(pos).cuda()
    val, grad, hess, _ = t.eval(dpos, mode=blip.VGH)
    v2, g2, lap, _ = t.eval(dpos, mode=blip.VGL)
    torch.cuda.synchronize()
    tv, tg, tl = tolerances(A, grid, float(np.abs(c).max()))
    assert hess.shape == (M, 6, L)
    assert float((hess[:, 0] + hess[:, 1] + hess[:, 2] - lap).abs().max()) <= 4 * tl
    assert float((val - v2).abs().max()) <= 2 * tv and float((grad - g2).abs().max()) <= 2 * tg
    t.close()


def test_hessian_non_finite_errors_and_host_entry(torch_cuda, blip):
    torch = torch_cuda
    grid, L = (8, 8, 8), 12
    A, c, pos = workloads.small_case(grid, L, 40, TRICLINIC, seed=2)
    pos[3, 0] = np.inf
    t = blip.BlipTable(A, grid, L, c)
    for dtype in ("f32", "f64"):
        val, grad, hess, cell = run_vgh(torch, blip, t, pos, L, dtype)
        assert np.isnan(val[3]).all() and np.isnan(grad[3]).all() and np.isnan(hess[3]).all() and (cell[3] == -1).all()
        good = np.arange(40) != 3
        check(A, grid, c, pos[good], (val[good], grad[good], hess[good], cell[good]), dtype)
    lib = blip.lib()
    assert lib.blipgpu_eval(t.handle, None, 4, blip.VGH, None, None, None, 12, None, None) == blip.EINVAL
    assert lib.blipgpu_eval(t.handle, None, 4, 3, None, None, None, 12, None, None) == blip.EINVAL       # unknown mode
    assert lib.blipgpu_eval_contract(t.handle, None, 4, blip.VGH, None, 12, None, None, None) == blip.EINVAL
    # host buffers
    good = np.arange(40) != 3
    hpos = np.ascontiguousarray(pos[good])
    M = hpos.shape[0]
    hval = np.empty((M, 12), dtype=np.float32)
    hgrad = np.empty((M, 3, 12), dtype=np.float32)
    hhess = np.empty((M, 6, 12), dtype=np.float32)
    hcell = np.empty((M, 3), dtype=np.int32)
    blip.blipgpu_eval_host(t.handle, hpos, M, blip.VGH, hval, hgrad, hhess, 12, hcell)
    check(A, grid, c, hpos, (hval, hgrad, hhess, hcell), "f32")
    t.close()


def test_hessian_tio2_one_walker(torch_cuda, blip):
    """The local-energy call of the paper's largest system: one walker (1,536 positions) of the
    TiO2 config, 768 orbitals, fp32 and fp64, every output."""
    cfg = workloads.CONFIGS["tio2"]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    pos = workloads.positions(cfg, M=cfg.electrons)
    t = blip.BlipTable(A, cfg.grid, cfg.norb, c)
    worst = check(A, cfg.grid, c, pos, run_vgh(torch_cuda, blip, t, pos, cfg.norb, "f32"), "f32")
    assert worst.max() < 0.5, worst
    check(A, cfg.grid, c, pos, run_vgh(torch_cuda, blip, t, pos, cfg.norb, "f64"), "f64")
    t.close()
