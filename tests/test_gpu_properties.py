"""Properties that hold at any size, checked on EVERY output of the full-size configurations in
the launch configuration bench.py times (the element-by-element comparisons with the oracle are
in test_gpu_parity.py):

* partition of unity: a constant table c = kappa gives psi = kappa, grad = 0, lap = 0 everywhere
  (the 4 cubic B-spline weights sum to 1, their derivatives to 0; reading R2).  It sees
  a wrong WEIGHT; it cannot see a wrong row or plane (all rows are equal);
* linear exactness: c[k][l] = alpha_l + sum_a beta_al k_a gives psi_l = alpha_l + sum_a beta_al t_a,
  grad = sum_a beta_al J[a][.], lap = 0 wherever the 4x4x4 block does not cross the periodic seam
  (first moment of the cubic B-spline; the closed form of tests/test_oracle_pins.py).  Every row
  of the table differs from its neighbours and every orbital has its own ramp, so a wrong row, a
  stale plane, a wrong halo or a wrong orbital column shifts the value by a whole beta;
* lattice periodicity: r and r + m1 a1 + m2 a2 + m3 a3 give the same orbitals.
"""
import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import tolerances, torch_cuda, blip  # noqa: F401 (fixtures)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,path", [("tio2", 5), ("tio2", 2), ("large", 1), ("small", 3)])
def test_partition_of_unity_full_size(torch_cuda, blip, name, path):
    torch = torch_cuda
    cfg = workloads.CONFIGS[name]
    A = workloads.lattice(cfg)
    kappa = 1.75
    c = torch.full((*cfg.grid, cfg.norb), kappa, dtype=torch.float32, device="cuda")     # built on the device
    h = blip.blipgpu_create(A, cfg.grid, cfg.norb, c)
    del c
    if path == 2:
        blip.blipgpu_set_tuning(h, 2, 0)                     # the FP32-pipe staged kernel (automatic: tensor cores, path 5)
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


@pytest.mark.parametrize("name,path", [("tio2", 5), ("tio2", 2), ("tio2", 1), ("small", 3)])
def test_linear_ramp_table_full_size(torch_cuda, blip, name, path):
    """Ramp table (see module docstring) on every position of the config whose block of sites stays
    clear of the periodic seam, against the closed form evaluated here in fp64."""
    torch = torch_cuda
    cfg = workloads.CONFIGS[name]
    A = workloads.lattice(cfg)
    n = np.array(cfg.grid)
    L = cfg.norb
    rng = np.random.default_rng(31)
    alpha = rng.integers(-16, 17, size=L) / 8.0             # dyadic: every table entry is exact in fp32
    beta = rng.integers(-8, 9, size=(3, L)) / 8.0
    k1 = torch.arange(n[0], device="cuda", dtype=torch.float32)[:, None, None, None]
    k2 = torch.arange(n[1], device="cuda", dtype=torch.float32)[None, :, None, None]
    k3 = torch.arange(n[2], device="cuda", dtype=torch.float32)[None, None, :, None]
    tb = torch.from_numpy(beta.astype(np.float32)).cuda()
    c = (torch.from_numpy(alpha.astype(np.float32)).cuda() + k1 * tb[0] + k2 * tb[1] + k3 * tb[2]).contiguous()
    cmax = float(c.abs().max())
    h = blip.blipgpu_create(A, cfg.grid, L, c)
    del c
    blip.blipgpu_set_tuning(h, path if path != 3 else 0, 0)
    hpos = workloads.positions(cfg)
    pos = torch.from_numpy(hpos).cuda()
    M = pos.shape[0]
    val = torch.empty((M, L), dtype=torch.float32, device="cuda")
    grad = torch.empty((M, 3, L), dtype=torch.float32, device="cuda")
    lap = torch.empty((M, L), dtype=torch.float32, device="cuda")
    cell = torch.empty((M, 3), dtype=torch.int32, device="cuda")
    blip.blipgpu_eval(h, pos, M, blip.VGL, val, grad, lap, L, cell)
    torch.cuda.synchronize()
    assert blip.blipgpu_last_path(h) == path
    blip.blipgpu_destroy(h)
    # closed form, fp64, from the definition of the grid coordinate t = n * frac(r . A^-1)
    G = np.linalg.inv(A)
    u = hpos @ G
    t = (u - np.floor(u)) * n
    i = cell.cpu().numpy().astype(np.int64)                  # (bit-exactness against the oracle is tested elsewhere)
    f = t - i
    f -= n * np.round(f / n)                                 # a position within rounding of the seam
    assert f.min() > -1e-9 and f.max() < 1 + 1e-9
    interior = ((i >= 1) & (i <= n - 3)).all(axis=1)
    assert interior.mean() > 0.8
    J = (G * n).T                                            # J[a][i] = n_a G[i][a]
    ref_val = alpha[None, :] + t @ beta
    ref_grad = np.einsum("ai,al->il", J, beta)               # the same for every position
    tv, tg, tl = tolerances(A, cfg.grid, cmax)
    ok = torch.from_numpy(interior).cuda()
    assert float((val.double() - torch.from_numpy(ref_val).cuda()).abs()[ok].max()) <= tv
    assert float((grad.double() - torch.from_numpy(ref_grad).cuda()[None]).abs()[ok].max()) <= tg
    assert float(lap.abs()[ok].max()) <= tl
