"""Parity of the CUDA path (through the C ABI) against the CPU fp64 oracle, on a B200.

Tolerances are BASELINE.json north_star's: value <= 2e-5 max|c|, gradient <= 2e-5 max|c| / h,
Laplacian <= 5e-5 max|c| / h^2 with h the largest grid-plane spacing (reading R13),
max-norm over positions, orbitals and components; cell indices bit-exact.
"""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

VAL_TOL, GRAD_TOL, LAP_TOL = 2e-5, 2e-5, 5e-5


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    torch.cuda.set_device(0)
    return torch


@pytest.fixture(scope="module")
def blip():
    import paper_1204_1121_b200 as b
    b.lib()
    return b


def tolerances(A, grid, cmax):
    h = float(oracle.spacing(A, grid).max())
    return VAL_TOL * cmax, GRAD_TOL * cmax / h, LAP_TOL * cmax / (h * h)


def run_gpu(torch, blip, A, grid, c, pos, mode=1, ld=None, want_cell=True, table=None):
    L = c.shape[3]
    own = table is None
    if own:
        table = blip.BlipTable(A, grid, L, c)
    if ld is not None:
        table.ld = ld
    dpos = torch.from_numpy(np.ascontiguousarray(pos)).cuda()
    val, grad, lap, cell = table.eval(dpos, mode=mode, want_cell=want_cell)
    torch.cuda.synchronize()
    out = (val.cpu().numpy(), None if grad is None else grad.cpu().numpy(),
           None if lap is None else lap.cpu().numpy(), None if cell is None else cell.cpu().numpy())
    if own:
        table.close()
    return out


def compare(A, grid, c, pos, gpu, mode=1, cmax=None, report=None):
    val, grad, lap, cell = gpu
    oval, ograd, olap, ocell = oracle.eval_fast(A, grid, c, pos, mode=mode)
    cmax = float(np.abs(c).max()) if cmax is None else cmax
    tv, tg, tl = tolerances(A, grid, cmax)
    if cell is not None:
        assert np.array_equal(cell, ocell), "cell indices must be bit-exact"
    ev = float(np.abs(val - oval).max()) if val.size else 0.0
    assert ev <= tv, f"value error {ev:.3e} > {tv:.3e}"
    if mode == 1:
        eg = float(np.abs(grad - ograd).max()) if grad.size else 0.0
        el = float(np.abs(lap - olap).max()) if lap.size else 0.0
        assert eg <= tg, f"gradient error {eg:.3e} > {tg:.3e}"
        assert el <= tl, f"Laplacian error {el:.3e} > {tl:.3e}"
        if report is not None:
            report.update(val=ev / tv, grad=eg / tg, lap=el / tl)


# ------------------------------------------------------------------ config 1 and 2, in full
@pytest.mark.parametrize("name", ["tiny", "small"])
def test_config_full(torch_cuda, blip, name):
    cfg = workloads.CONFIGS[name]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    pos = workloads.positions(cfg)
    rep = {}
    compare(A, cfg.grid, c, pos, run_gpu(torch_cuda, blip, A, cfg.grid, c, pos), report=rep)
    assert max(rep.values()) < 0.5, rep          # expected ~1-5 % of the tolerances
    compare(A, cfg.grid, c, pos, run_gpu(torch_cuda, blip, A, cfg.grid, c, pos, mode=0), mode=0)


# ------------------------------------------------------------------ config 3 and 4 (TiO2-sized)
@pytest.fixture(scope="module")
def tio2(torch_cuda, blip):
    cfg = workloads.CONFIGS["tio2"]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    table = blip.BlipTable(A, cfg.grid, cfg.norb, c)
    yield cfg, A, c, table
    table.close()


def test_config_tio2_full_size_sampled(torch_cuda, blip, tio2):
    """Full 49,152-position call in the bench's launch configuration; cells checked for every
    position, val/grad/lap on a seeded sample of positions the oracle computes one by one."""
    cfg, A, c, table = tio2
    pos = workloads.positions(cfg)
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, cfg.grid, c, pos, table=table)
    assert blip.blipgpu_last_path(table.handle) == 2        # the staged kernel, as in bench.py
    ocell, _ = oracle.cellmap(A, cfg.grid, pos)
    assert np.array_equal(cell, ocell)
    rng = np.random.default_rng(99)
    pick = np.sort(rng.choice(pos.shape[0], size=3000, replace=False))
    pick[:200] = np.arange(0, 1000, 5)                 # make sure clustered ones are in
    compare(A, cfg.grid, c, pos[pick], (val[pick], grad[pick], lap[pick], cell[pick]))
    # value-only mode at full size
    val0, _, _, _ = run_gpu(torch_cuda, blip, A, cfg.grid, c, pos, mode=0, table=table, want_cell=False)
    compare(A, cfg.grid, c, pos[pick], (val0[pick], None, None, None), mode=0)


@pytest.mark.parametrize("M", [1, 8, 32, 128, 512, 1536])
@pytest.mark.parametrize("mode", [0, 1])
def test_config_sweep(torch_cuda, blip, tio2, M, mode):
    cfg, A, c, table = tio2
    pos = workloads.positions(cfg, M=M)
    compare(A, cfg.grid, c, pos, run_gpu(torch_cuda, blip, A, cfg.grid, c, pos, mode=mode, table=table),
            mode=mode)
    assert blip.blipgpu_last_path(table.handle) == 3        # the split kernel


# ------------------------------------------------------------------ config 5 (6.3 GB, triclinic)
def test_config_large_full_size_sampled(torch_cuda, blip):
    cfg = workloads.CONFIGS["large"]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    pos = workloads.positions(cfg)
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, cfg.grid, c, pos)
    ocell, _ = oracle.cellmap(A, cfg.grid, pos)
    assert np.array_equal(cell, ocell)
    pick = np.sort(np.random.default_rng(98).choice(pos.shape[0], size=1500, replace=False))
    rep = {}
    compare(A, cfg.grid, c, pos[pick], (val[pick], grad[pick], lap[pick], cell[pick]), report=rep)
    assert max(rep.values()) < 0.5, rep
