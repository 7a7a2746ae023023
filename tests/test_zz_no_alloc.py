"""blipgpu_eval_static — the entry point for callers that may not allocate device memory while they
sample — against blipgpu_eval, the path every other GPU test covers.

Who needs it: a QMC host code that has handed the rest of the GPU's memory to its own arena after
set-up (a later cudaMalloc from inside a library fails there), or one that keeps walkers running on
other streams (cudaMalloc / cudaFree stall the whole device until they drain).  blipgpu_eval grows
its grouping workspace with cudaMalloc on demand; blipgpu_eval_static keeps that workspace in a
fixed 768 KiB array inside libblipgpu.so, takes at most 65,536 positions and 32,768 cell bricks per
call, and refuses anything larger with BLIPGPU_ELIMIT.

What is checked here: the same outputs as blipgpu_eval within the tolerances the parity tests use
(BASELINE.json north_star: 2e-5 max|c| on values, 2e-5 max|c| / h on gradients, 5e-5 max|c| / h^2
on Laplacians; cell indices bit-exact), on two calls in a row — the fixed array is shared by all
calls and keeps what the last one left, so the second call, smaller and on other positions, is the
one that would show a missing clear.  Also: two tables taking turns on the array, the largest
batch the array allows, and the refusals.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this
outside-§8 entry point must not hide the parity tests.  Every test builds its own tables, so the
file passes alone in a fresh process (where its first call does the per-device address look-up) and
at the end of the whole suite alike.
"""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

VAL_TOL, GRAD_TOL, LAP_TOL = 2e-5, 2e-5, 5e-5          # as tests/test_gpu_parity.py
TRICLINIC = ((20, 0, 0), (3, 19, 0), (2, 2, 24))


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


def outputs(torch, M, ld, mode):
    val = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda")          # 7: never a result of these tables
    grad = torch.full((M, 3, ld), 7.0, dtype=torch.float32, device="cuda") if mode == 1 else None
    lap = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda") if mode == 1 else None
    cell = torch.full((M, 3), -7, dtype=torch.int32, device="cuda")
    return val, grad, lap, cell


def both_paths(torch, blip, table, pos, mode=1, path=0):
    """(existing path, allocation-free path) outputs as numpy, columns 0..L-1."""
    M, ld, L = pos.shape[0], table.ld, table.norb
    dpos = torch.from_numpy(np.ascontiguousarray(pos)).cuda()
    ref = outputs(torch, M, ld, mode)
    new = outputs(torch, M, ld, mode)
    blip.blipgpu_set_tuning(table.handle, path, 0)
    blip.blipgpu_eval(table.handle, dpos, M, mode, ref[0], ref[1], ref[2], ld, ref[3])
    blip.blipgpu_set_tuning(table.handle, 0, 0)
    blip.blipgpu_eval_static(table.handle, dpos, M, mode, new[0], new[1], new[2], ld, new[3])
    torch.cuda.synchronize()
    cut = lambda x: None if x is None else x.cpu().numpy()[..., :L]
    return ([cut(ref[0]), cut(ref[1]), cut(ref[2]), ref[3].cpu().numpy()],
            [cut(new[0]), cut(new[1]), cut(new[2]), new[3].cpu().numpy()])


def assert_same(A, grid, c, ref, new, mode=1, exact=False):
    cmax = float(np.abs(c).max())
    h = float(oracle.spacing(A, grid).max())
    tols = (VAL_TOL * cmax, GRAD_TOL * cmax / h, LAP_TOL * cmax / (h * h))
    assert np.array_equal(new[3], ref[3]), "cell indices must be bit-exact"
    for k, name in enumerate(("value", "gradient", "Laplacian")[: 3 if mode == 1 else 1]):
        assert np.isfinite(new[k]).all(), name
        if exact:
            assert np.array_equal(new[k], ref[k]), f"{name}: the direct kernel's bits"
        err = float(np.abs(new[k].astype(np.float64) - ref[k]).max())
        assert err <= tols[k], f"{name} differs from blipgpu_eval by {err:.3e} > {tols[k]:.3e}"


def test_two_calls_in_a_row_match_blipgpu_eval(torch_cuda, blip):
    """Call 1: 5,000 positions.  Call 2, straight after it on the same array: 1,800 other positions.
    Each against blipgpu_eval's automatic path, and bit for bit against its direct-gather kernel."""
    grid, L = (9, 10, 13), 130
    A, c, pos1 = workloads.small_case(grid, L, 5000, TRICLINIC, seed=11)
    _, _, pos2 = workloads.small_case(grid, L, 1800, TRICLINIC, seed=12)
    table = blip.BlipTable(A, grid, L, c)
    try:
        for pos in (pos1, pos2):
            ref, new = both_paths(torch_cuda, blip, table, pos)
            assert_same(A, grid, c, ref, new)
            assert blip.blipgpu_last_path(table.handle) == 1
            ref, new = both_paths(torch_cuda, blip, table, pos, path=1)
            assert_same(A, grid, c, ref, new, exact=True)
        # ... and the oracle has the last word on the second call (the one that ran on a used array)
        oval, ograd, olap, ocell = oracle.eval_fast(A, grid, c, pos2)
        assert_same(A, grid, c, [oval, ograd, olap, ocell], new)
    finally:
        table.close()


def test_two_tables_take_turns_on_the_shared_array(torch_cuda, blip):
    """The array belongs to the library, not to a handle: a table with many bricks, then one with few
    (its counts sit where the first table's were), then the first again; value-only mode in between.
    The second table's batch is dense, so blipgpu_eval answers it from its tensor-core kernel:
    different last bits, same tolerances."""
    gridA, LA = (24, 20, 28), 36                            # 6 x 5 x 7 = 210 bricks, diagonal lattice
    AA = np.diag([11.0, 9.5, 13.0])
    cA = np.random.default_rng(21).standard_normal((*gridA, LA)).astype(np.float32)
    posA = (np.random.default_rng(22).random((7000, 3)) * 3.0 - 1.0) @ AA
    gridB, LB = (12, 12, 16), 256                           # 3 x 3 x 4 = 36 bricks, triclinic
    AB, cB, posB = workloads.small_case(gridB, LB, 6000, TRICLINIC, seed=23)
    tA = blip.BlipTable(AA, gridA, LA, cA)
    tB = blip.BlipTable(AB, gridB, LB, cB)
    try:
        ref, new = both_paths(torch_cuda, blip, tA, posA)
        assert_same(AA, gridA, cA, ref, new)
        ref, new = both_paths(torch_cuda, blip, tB, posB)
        assert_same(AB, gridB, cB, ref, new)
        ref, new = both_paths(torch_cuda, blip, tB, posB[:3000], mode=0)
        assert_same(AB, gridB, cB, ref, new, mode=0)
        ref, new = both_paths(torch_cuda, blip, tA, posA[::-1])
        assert_same(AA, gridA, cA, ref, new)
    finally:
        tA.close()
        tB.close()


def test_largest_batch_and_non_finite_positions(torch_cuda, blip):
    """Exactly BLIPGPU_STATIC_MAX_POSITIONS positions, some of them NaN / Inf: NaN outputs and
    cell = -1 for those, as blipgpu_eval documents, everything else as above."""
    grid, L = (16, 16, 16), 8
    M = blip.STATIC_MAX_POSITIONS
    A, c, pos = workloads.small_case(grid, L, M, np.diag([10.0, 10.0, 10.0]), seed=31)
    bad = np.arange(5, M, 4099)
    pos[bad, 1] = np.nan
    pos[bad[::2], 0] = np.inf
    table = blip.BlipTable(A, grid, L, c)
    try:
        ref, new = both_paths(torch_cuda, blip, table, pos)
        good = np.ones(M, dtype=bool)
        good[bad] = False
        assert (new[3][bad] == -1).all() and np.array_equal(new[3], ref[3])
        for k in range(3):
            assert np.isnan(new[k][bad]).all()
        assert_same(A, grid, c, [ref[0][good], ref[1][good], ref[2][good], ref[3][good]],
                    [new[0][good], new[1][good], new[2][good], new[3][good]])
    finally:
        table.close()


def test_refusals_are_clear_and_allocate_nothing(torch_cuda, blip):
    """One position too many, a table with too many bricks, the Hessian mode: error codes, nothing
    launched, outputs untouched; M = 0 is fine.  And the device's memory in use does not move across
    calls of any size (the point of the entry point)."""
    torch = torch_cuda
    grid, L = (8, 8, 8), 4
    A, c, pos = workloads.small_case(grid, L, 64, np.diag([5.0, 5.0, 5.0]), seed=41)
    table = blip.BlipTable(A, grid, L, c)
    big = None
    try:
        M = blip.STATIC_MAX_POSITIONS + 1
        dpos = torch.zeros((M, 3), dtype=torch.float64, device="cuda")
        val, grad, lap, cell = outputs(torch, M, table.ld, 1)
        launches = blip.blipgpu_launch_count(table.handle)
        with pytest.raises(blip.BlipGpuError) as ei:
            blip.blipgpu_eval_static(table.handle, dpos, M, blip.VGL, val, grad, lap, table.ld, cell)
        assert ei.value.code == blip.ELIMIT and "blipgpu_eval_static" in str(ei.value) and "too large" in str(ei.value)
        with pytest.raises(blip.BlipGpuError) as ei:
            blip.blipgpu_eval_static(table.handle, dpos, 64, blip.VGH, val, grad, lap, table.ld, cell)
        assert ei.value.code == blip.EINVAL
        blip.blipgpu_eval_static(table.handle, dpos, 0, blip.VGL, val, grad, lap, table.ld, cell)
        torch.cuda.synchronize()
        assert blip.blipgpu_launch_count(table.handle) == launches
        assert float(val.min()) == 7.0 and float(val.max()) == 7.0 and int(cell.max()) == -7

        gbig = (132, 128, 128)                              # 33 x 32 x 32 = 33,792 bricks > 32,768
        big = blip.BlipTable(np.diag([30.0, 29.0, 29.0]), gbig, 1, np.zeros((*gbig, 1), dtype=np.float32))
        v1, g1, l1, c1 = outputs(torch, 64, big.ld, 1)
        with pytest.raises(blip.BlipGpuError) as ei:
            blip.blipgpu_eval_static(big.handle, dpos, 64, blip.VGL, v1, g1, l1, big.ld, c1)
        assert ei.value.code == blip.ELIMIT

        # no allocation whatever the batch: bytes in use on the device before and after a run of calls of
        # growing size on a fresh handle (blipgpu_eval would have grown its workspace at 4,096 positions)
        fresh = blip.BlipTable(A, grid, L, c)
        try:
            batches = [torch.from_numpy(workloads.small_case(grid, L, m, np.diag([5.0, 5.0, 5.0]), seed=m)[2]).cuda()
                       for m in (64, 4096, 30000)]
            outs = [outputs(torch, b.shape[0], fresh.ld, 1) for b in batches]
            blip.blipgpu_eval_static(fresh.handle, batches[0], 64, blip.VGL, *outs[0][:3], fresh.ld, outs[0][3])
            torch.cuda.synchronize()
            free0, _ = torch.cuda.mem_get_info()
            for b, o in zip(batches, outs):
                blip.blipgpu_eval_static(fresh.handle, b, b.shape[0], blip.VGL, o[0], o[1], o[2], fresh.ld, o[3])
            torch.cuda.synchronize()
            free1, _ = torch.cuda.mem_get_info()
            assert free1 == free0, (free0, free1)
        finally:
            fresh.close()
    finally:
        table.close()
        if big is not None:
            big.close()
