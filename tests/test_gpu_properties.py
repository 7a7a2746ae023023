"""Properties that hold at any size, checked on EVERY output of the full-size configurations in
the launch configuration bench.py times (the sampled comparisons with the oracle are in
test_gpu_parity.py):

* partition of unity: a constant table c = kappa gives psi = kappa, grad = 0, lap = 0 everywhere
  (the 4 cubic B-spline weights sum to 1, their derivatives to 0; reading R2) — any
  wrong row, plane, halo or weight in any kernel breaks it;
* lattice periodicity: r and r + m1 a1 + m2 a2 + m3 a3 give the same orbitals.
"""
import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import tolerances, torch_cuda, blip  # noqa: F401 (fixtures)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,path", [("tio2", 2), ("large", 1), ("small", 3)])
def test_partition_of_unity_full_size(torch_cuda, blip, name, path):
    torch = torch_cuda
    cfg = workloads.CONFIGS[name]
    A = workloads.lattice(cfg)
    kappa = 1.75
    c = torch.full((*cfg.grid, cfg.norb), kappa, dtype=torch.float32, device="cuda")     # built on the device
    h = blip.blipgpu_create(A, cfg.grid, cfg.norb, c)
    del c
    pos = torch.from_numpy(workloads.positions(cfg)).cuda()
    M, L = pos.shape[0], cfg.norb
    val = torch.empty((M, L), dtype=torch.float32, device="cuda")
    grad = torch.empty((M, 3, L), dtype=torch.float32, device="cuda")
    lap = torch.empty((M, L), dtype=torch.float32, device="cuda")
    blip.blipgpu_eval(h, pos, M, blip.VGL, val, grad, lap, L)
    torch.cuda.synchronize()
    assert blip.blipgpu_last_path(h) == path
    tv, tg, tl = tolerances(A, cfg.grid, kappa)
    assert float((val - kappa).abs().max()) <= tv
    assert float(grad.abs().max()) <= tg
    assert float(lap.abs().max()) <= tl
    blip.blipgpu_destroy(h)


def test_periodicity_full_size_tio2(torch_cuda, blip):
    torch = torch_cuda
    cfg = workloads.CONFIGS["tio2"]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    cmax = float(np.abs(c).max())
    t = blip.BlipTable(A, cfg.grid, cfg.norb, c)
    pos = workloads.positions(cfg)
    shift = np.random.default_rng(12).integers(-3, 4, size=(pos.shape[0], 3)).astype(np.float64) @ A
    out = []
    for p in (pos, pos + shift):
        val, grad, lap, cell = t.eval(torch.from_numpy(np.ascontiguousarray(p)).cuda(), mode=blip.VGL, want_cell=True)
        torch.cuda.synchronize()
        out.append((val, grad, lap, cell))
    tv, tg, tl = tolerances(A, cfg.grid, cmax)
    # the shifted position lands in the same cell except within rounding of a cell face; the
    # spline is C^2 there, so values still agree (reading R10)
    same = (out[0][3] == out[1][3]).all(dim=1).float().mean().item()
    assert same > 0.999
    assert float((out[0][0] - out[1][0]).abs().max()) <= 2 * tv
    assert float((out[0][1] - out[1][1]).abs().max()) <= 2 * tg
    assert float((out[0][2] - out[1][2]).abs().max()) <= 2 * tl
    t.close()
