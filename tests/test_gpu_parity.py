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


def compare_all(A, grid, c, pos, gpu, mode=1, chunk=8192):
    """Every output of a full-size call against the oracle ("all positions x orbitals
    of each config"), chunk by chunk to bound the fp64 reference in host memory.  Returns the
    largest error of each quantity as a fraction of its tolerance."""
    val, grad, lap, cell = gpu
    cmax = float(np.abs(c).max())
    tv, tg, tl = tolerances(A, grid, cmax)
    worst = {"val": 0.0, "grad": 0.0, "lap": 0.0}
    for lo in range(0, pos.shape[0], chunk):
        hi = min(lo + chunk, pos.shape[0])
        oval, ograd, olap, ocell = oracle.eval_fast(A, grid, c, pos[lo:hi], mode=mode)
        if cell is not None:
            assert np.array_equal(cell[lo:hi], ocell), "cell indices must be bit-exact"
        worst["val"] = max(worst["val"], float(np.abs(val[lo:hi] - oval).max()) / tv)
        if mode == 1:
            worst["grad"] = max(worst["grad"], float(np.abs(grad[lo:hi] - ograd).max()) / tg)
            worst["lap"] = max(worst["lap"], float(np.abs(lap[lo:hi] - olap).max()) / tl)
    assert worst["val"] <= 1.0 and worst["grad"] <= 1.0 and worst["lap"] <= 1.0, worst
    return worst


def test_config_tio2_full_size_every_output(torch_cuda, blip, tio2):
    """The full 49,152-position call in the launch configuration bench.py times (the staged kernel
    on the tensor cores): cells and val / grad / lap of EVERY position and orbital against the
    oracle, both modes; then the same for the FP32-pipe staged kernel."""
    cfg, A, c, table = tio2
    pos = workloads.positions(cfg)
    gpu = run_gpu(torch_cuda, blip, A, cfg.grid, c, pos, table=table)
    assert blip.blipgpu_last_path(table.handle) == 5        # the tensor-core staged kernel, as in bench.py
    worst = compare_all(A, cfg.grid, c, pos, gpu)
    assert max(worst.values()) < 0.5, worst                 # expected a few % of the tolerances
    val0, _, _, _ = run_gpu(torch_cuda, blip, A, cfg.grid, c, pos, mode=0, table=table, want_cell=False)
    compare_all(A, cfg.grid, c, pos, (val0, None, None, None), mode=0)
    try:
        blip.blipgpu_set_tuning(table.handle, path=2)
        gpu = run_gpu(torch_cuda, blip, A, cfg.grid, c, pos, table=table)
        assert blip.blipgpu_last_path(table.handle) == 2
        worst = compare_all(A, cfg.grid, c, pos, gpu)
        assert max(worst.values()) < 0.5, worst
    finally:
        blip.blipgpu_set_tuning(table.handle, path=0)


def test_tio2_full_size_staged_equals_direct_and_is_repeatable(torch_cuda, blip, tio2):
    """At full size: the staged kernel (persistent CTAs, TMA ring, mbarrier hand-offs) returns the
    bits of the direct kernel on every output, and 20 repeated calls return the bits of the first
    one (a stale plane or a lost hand-off would show as a flicker)."""
    torch = torch_cuda
    cfg, A, c, table = tio2
    dpos = torch.from_numpy(workloads.positions(cfg)).cuda()
    M, ld = dpos.shape[0], table.ld

    def call():
        val = torch.empty((M, ld), dtype=torch.float32, device="cuda")
        grad = torch.empty((M, 3, ld), dtype=torch.float32, device="cuda")
        lap = torch.empty((M, ld), dtype=torch.float32, device="cuda")
        blip.blipgpu_eval(table.handle, dpos, M, blip.VGL, val, grad, lap, ld)
        return val, grad, lap

    try:
        blip.blipgpu_set_tuning(table.handle, path=2)
        first = call()
        assert blip.blipgpu_last_path(table.handle) == 2
        for _ in range(20):
            again = call()
            torch.cuda.synchronize()
            for a, b in zip(first, again):
                assert torch.equal(a, b)
            del again
        blip.blipgpu_set_tuning(table.handle, path=1)
        direct = call()
        torch.cuda.synchronize()
        assert blip.blipgpu_last_path(table.handle) == 1
        for a, b in zip(first, direct):
            assert torch.equal(a, b)
    finally:
        blip.blipgpu_set_tuning(table.handle, path=0)


@pytest.mark.parametrize("M", [1, 8, 32, 128, 512, 1536])
@pytest.mark.parametrize("mode", [0, 1])
def test_config_sweep(torch_cuda, blip, tio2, M, mode):
    cfg, A, c, table = tio2
    pos = workloads.positions(cfg, M=M)
    compare(A, cfg.grid, c, pos, run_gpu(torch_cuda, blip, A, cfg.grid, c, pos, mode=mode, table=table),
            mode=mode)
    assert blip.blipgpu_last_path(table.handle) == 3        # the split kernel


# ------------------------------------------------------------------ config 5 (6.3 GB, triclinic)
def test_config_large_full_size_every_output(torch_cuda, blip):
    """24,576 positions x 1,536 orbitals on the 6.3 GB triclinic table (grouped direct kernel, as
    bench.py --workload large runs it): every output against the oracle."""
    cfg = workloads.CONFIGS["large"]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    pos = workloads.positions(cfg)
    t = blip.BlipTable(A, cfg.grid, cfg.norb, c)
    gpu = run_gpu(torch_cuda, blip, A, cfg.grid, c, pos, table=t)
    assert blip.blipgpu_last_path(t.handle) == 1
    t.close()
    worst = compare_all(A, cfg.grid, c, pos, gpu, chunk=4096)
    assert max(worst.values()) < 0.5, worst
