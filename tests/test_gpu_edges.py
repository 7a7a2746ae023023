"""Edge cases of the CUDA path against the oracle: ragged orbital counts, padded pitch, empty
batch, wrap-everywhere grids, grids that are not a multiple of the grouping brick, far-away
and non-finite positions, adversarial cell-index inputs, the host-buffer entry point, and
argument errors."""
import ctypes

import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import compare, run_gpu, tolerances, torch_cuda, blip  # noqa: F401 (fixtures)

pytestmark = pytest.mark.gpu

TRICLINIC = ((20.0, 0.0, 0.0), (3.0, 19.0, 0.0), (2.0, 2.0, 24.0))
SKEW = ((5.0, 0.3, -0.2), (1.1, 4.0, 0.7), (-0.6, 0.9, 6.0))


@pytest.mark.parametrize("L", [1, 3, 5, 33, 130, 257])
def test_ragged_orbital_counts(torch_cuda, blip, L):
    A, c, pos = workloads.small_case((6, 5, 7), L, 300, SKEW, seed=L, spread=4.0)
    for mode in (0, 1):
        compare(A, (6, 5, 7), c, pos, run_gpu(torch_cuda, blip, A, (6, 5, 7), c, pos, mode=mode), mode=mode)


def test_wider_output_pitch(torch_cuda, blip):
    A, c, pos = workloads.small_case((8, 8, 8), 10, 100, TRICLINIC, seed=2)
    compare(A, (8, 8, 8), c, pos, run_gpu(torch_cuda, blip, A, (8, 8, 8), c, pos, ld=24))


def test_empty_batch(torch_cuda, blip):
    A, c, pos = workloads.small_case((4, 4, 4), 4, 1, SKEW, seed=2)
    t = blip.BlipTable(A, (4, 4, 4), 4, c)
    n0 = t.launch_count()
    val, grad, lap, cell = t.eval(torch_cuda.empty((0, 3), dtype=torch_cuda.float64, device="cuda"))
    assert val.shape == (0, 4) and t.launch_count() == n0
    t.close()


@pytest.mark.parametrize("grid", [(4, 4, 4), (5, 7, 9), (4, 13, 6)])
@pytest.mark.parametrize("M", [700, 5000])
def test_wrap_everywhere_and_non_brick_grids(torch_cuda, blip, grid, M):
    """4x4x4: every block of 64 sites wraps.  M = 5000 goes through the grouping path with
    grids that are not a multiple of the 4-cell brick."""
    A, c, pos = workloads.small_case(grid, 12, M, TRICLINIC, seed=M, spread=6.0)
    compare(A, grid, c, pos, run_gpu(torch_cuda, blip, A, grid, c, pos))


def test_grouped_equals_ungrouped(torch_cuda, blip):
    """The same positions evaluated in one grouped call (M > threshold) and in small
    ungrouped calls give bit-identical results: caller order is preserved."""
    A, c, pos = workloads.small_case((12, 9, 10), 40, 6000, SKEW, seed=8, spread=2.0)
    t = blip.BlipTable(A, (12, 9, 10), 40, c)
    full = run_gpu(torch_cuda, blip, A, (12, 9, 10), c, pos, table=t)
    for lo in range(0, 6000, 1500):
        part = run_gpu(torch_cuda, blip, A, (12, 9, 10), c, pos[lo:lo + 1500], table=t)
        for a, b in zip(full, part):
            assert np.array_equal(a[lo:lo + 1500], b)
    t.close()


# ------------------------------------------------------------------ staged (TMA / shared memory) path
STAGED_CASES = [((9, 10, 13), 130, 3000, TRICLINIC), ((20, 7, 8), 128, 1200, SKEW),
                ((17, 12, 19), 257, 9000, TRICLINIC), ((4, 4, 8), 200, 700, SKEW)]


@pytest.mark.parametrize("grid,L,M,lat", STAGED_CASES)
def test_staged_path_matches_oracle_and_direct_path(torch_cuda, blip, grid, L, M, lat):
    """The staged kernel forced on grids that are ragged against the 4x4 pencil cross-section,
    orbital counts that are not a multiple of the 128-orbital tile, and
    pencils without electrons: parity with the oracle, and bit-identical to the direct kernel."""
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=L + M, spread=3.0)
    t = blip.BlipTable(A, grid, L, c)
    for mode in (1, 0):
        blip.blipgpu_set_tuning(t.handle, path=2)
        n0 = t.launch_count()
        staged = run_gpu(torch_cuda, blip, A, grid, c, pos, mode=mode, table=t)
        assert t.launch_count() - n0 == 2                # grouping (one cooperative launch), staged eval
        compare(A, grid, c, pos, staged, mode=mode)
        blip.blipgpu_set_tuning(t.handle, path=1)
        direct = run_gpu(torch_cuda, blip, A, grid, c, pos, mode=mode, table=t)
        for a, b in zip(staged, direct):
            assert (a is None and b is None) or np.array_equal(a, b)
    t.close()


def test_axis_aligned_lattice_mode(torch_cuda, blip):
    """Lattice vectors along the Cartesian axes select the kernels' MODE 2 (diagonal J): staged,
    direct and split kernels against the oracle, staged and direct bit-identical."""
    grid, L, M = (11, 9, 14), 140, 5000
    lat = ((7.0, 0.0, 0.0), (0.0, 8.5, 0.0), (0.0, 0.0, 9.25))
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=5, spread=2.0)
    t = blip.BlipTable(A, grid, L, c)
    out = {}
    for path in (2, 1):
        blip.blipgpu_set_tuning(t.handle, path=path)
        out[path] = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
        assert blip.blipgpu_last_path(t.handle) == path
        compare(A, grid, c, pos, out[path])
    for a, b in zip(out[2], out[1]):
        assert np.array_equal(a, b)
    blip.blipgpu_set_tuning(t.handle, path=0)             # automatic: dense batch -> staged (tensor cores), small batch -> split
    compare(A, grid, c, pos, run_gpu(torch_cuda, blip, A, grid, c, pos, table=t))
    assert blip.blipgpu_last_path(t.handle) == 5
    compare(A, grid, c, pos[:150], run_gpu(torch_cuda, blip, A, grid, c, pos[:150], table=t))
    assert blip.blipgpu_last_path(t.handle) == 3
    t.close()


def test_staged_path_with_more_work_items_than_the_sorter_takes(torch_cuda, blip):
    """93 x 93 pencils (> 8,192 work items): the scan kernel leaves the items in id order and
    the staged kernel skips the empty ones."""
    grid, L, M = (4, 372, 372), 128, 20000
    lat = ((3.0, 0.0, 0.0), (0.4, 90.0, 0.0), (0.1, 0.2, 95.0))
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=21, spread=1.0)
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_tuning(t.handle, path=2)
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
    assert blip.blipgpu_last_path(t.handle) == 2
    ocell, _ = oracle.cellmap(A, grid, pos)
    assert np.array_equal(cell, ocell)
    pick = np.arange(0, M, 7)
    compare(A, grid, c, pos[pick], (val[pick], grad[pick], lap[pick], cell[pick]))
    t.close()


def test_staged_path_clustered_and_non_finite(torch_cuda, blip):
    """All electrons in a few cells (long unit lists per plane, most pencils empty), plus
    non-finite positions, through the staged kernel."""
    grid, L = (24, 9, 17), 132
    A, c, pos = workloads.small_case(grid, L, 4000, TRICLINIC, seed=11, spread=0.02)
    pos[::7] += np.array(TRICLINIC[0]) * 0.37
    pos[5, 1] = np.nan
    pos[3999] = np.inf
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_tuning(t.handle, path=2)
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
    oval, ograd, olap, ocell = oracle.eval_fast(A, grid, c, pos)
    assert np.array_equal(cell, ocell)
    bad = np.isnan(oval).all(axis=1)
    assert bad.sum() == 2 and np.array_equal(np.isnan(val).all(axis=1), bad)
    assert np.isnan(grad[bad]).all() and np.isnan(lap[bad]).all()
    good = ~bad
    compare(A, grid, c, pos[good], (val[good], grad[good], lap[good], cell[good]))
    t.close()


def test_staged_path_unavailable_is_an_error(torch_cuda, blip):
    A, c, pos = workloads.small_case((6, 6, 6), 8, 10, SKEW, seed=4)      # fewer than 128 orbitals
    t = blip.BlipTable(A, (6, 6, 6), 8, c)
    assert blip.lib().blipgpu_set_tuning(t.handle, 2, 0) == blip.EINVAL
    assert blip.lib().blipgpu_set_tuning(t.handle, 3, 0) == blip.EINVAL
    assert blip.lib().blipgpu_set_tuning(t.handle, 1, 4) == blip.EINVAL
    assert blip.lib().blipgpu_set_tuning(t.handle, 1, 3) == blip.OK
    t.close()


def test_non_finite_positions(torch_cuda, blip):
    A, c, pos = workloads.small_case((6, 6, 6), 8, 3000, SKEW, seed=4)
    bad = [0, 17, 1500, 2999]
    pos[bad[0], 0] = np.nan
    pos[bad[1], 1] = np.inf
    pos[bad[2], 2] = -np.inf
    pos[bad[3]] = np.nan
    for M in (64, 3000):                      # ungrouped and grouped paths
        val, grad, lap, cell = run_gpu(torch_cuda, blip, A, (6, 6, 6), c, pos[:M])
        oval, ograd, olap, ocell = oracle.eval_fast(A, (6, 6, 6), c, pos[:M])
        assert np.array_equal(cell, ocell)
        nanrows = np.isnan(oval).all(axis=1)
        assert np.array_equal(np.isnan(val).all(axis=1), nanrows)
        assert np.isnan(grad[nanrows]).all() and np.isnan(lap[nanrows]).all()
        good = ~nanrows
        compare(A, (6, 6, 6), c, pos[:M][good], (val[good], grad[good], lap[good], cell[good]))


@pytest.mark.parametrize("path", [0, 1, 2, 5])
def test_overflow_on_a_single_axis(torch_cuda, blip, path):
    """Finite coordinates whose FRACTIONAL coordinate overflows on one axis only (sub-bohr lattice
    vectors, |r| near 1e308): the position is non-finite for the method — NaN outputs, cell = -1 on
    all three axes (include/blipgpu.h) — whichever axis it is and whichever kernel runs; its
    neighbours in the batch are unaffected."""
    grid, L = (12, 8, 12), 132
    lat = np.diag([0.5, 0.05, 0.5])
    A, c, pos = workloads.small_case(grid, L, 3000, lat, seed=13)
    bad = [3, 1000, 1001, 2999]
    pos[bad[0]] = (1.7e308, 0.01, 0.2)                       # axis 0 only
    pos[bad[1]] = (0.3, 1e308, 0.1)                          # axis 1 only
    pos[bad[2]] = (0.1, 0.02, -1.7e308)                      # axis 2 only
    pos[bad[3]] = (0.2, -1e307, 1.2e308)                     # axes 1 and 2
    assert np.isfinite(pos).all()
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_tuning(t.handle, path=path)
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
    assert blip.blipgpu_last_path(t.handle) == (path if path else 5)
    oval, ograd, olap, ocell = oracle.eval_fast(A, grid, c, pos)
    assert np.array_equal(cell, ocell) and (cell[bad] == -1).all()
    nanrows = np.isnan(oval).all(axis=1)
    assert nanrows.sum() == 4 and nanrows[bad].all()
    assert np.array_equal(np.isnan(val).all(axis=1), nanrows)
    assert np.isnan(grad[nanrows]).all() and np.isnan(lap[nanrows]).all()
    good = ~nanrows
    compare(A, grid, c, pos[good], (val[good], grad[good], lap[good], cell[good]))
    t.close()


def test_adversarial_cell_indices(torch_cuda, blip):
    """exact grid planes, denormal and tiny negative coordinates, +-1e3 cells, 1 ulp either
    side of a plane: GPU cell == oracle cell bit for bit."""
    lat = ((10.0, 0, 0), (0, 10.0, 0), (0, 0, 10.0))
    grid = (16, 16, 16)
    ks = np.arange(-40, 41, dtype=np.float64)
    planes = np.stack([ks * 0.625, ks * 0.625 + 0.3125, -ks * 0.625], axis=1)
    x = 0.625 * 5
    special = np.array([[-1e-300, 1e-300, -5e-324], [np.nextafter(x, 0), x, np.nextafter(x, 10)],
                        [1e4 + 0.1, -1e4 - 0.1, 6250.0], [-0.0, 0.0, 10.0],
                        [np.nextafter(10.0, 0), np.nextafter(10.0, 20), -10.0]])
    rng = np.random.default_rng(5)
    near = np.round(rng.random((2000, 3)) * 16) * 0.625 + rng.choice([-1, 0, 1], size=(2000, 3)) * 1e-15
    pos = np.concatenate([planes, special, near])
    c = workloads.coefficients(grid, 4)
    gpu = run_gpu(torch_cuda, blip, lat, grid, c, pos)
    compare(np.array(lat), grid, c, pos, gpu)
    # triclinic large grid, positions within a few ulp of cell faces in fractional space
    A = np.array(TRICLINIC)
    g2 = (96, 96, 112)
    u = rng.integers(0, 96, size=(3000, 3)) / np.array(g2) + rng.choice([-1, 0, 1], size=(3000, 3)) * 2e-16
    c2 = np.zeros((*g2, 1), dtype=np.float32)
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, g2, c2, u @ A)
    ocell, _ = oracle.cellmap(A, g2, u @ A)
    assert np.array_equal(cell, ocell)


def test_eval_host_matches_eval(torch_cuda, blip):
    torch = torch_cuda
    A, c, pos = workloads.small_case((10, 11, 9), 37, 20000, SKEW, seed=3)
    L, ld = 37, 40
    t = blip.BlipTable(A, (10, 11, 9), L, c)
    dev = run_gpu(torch, blip, A, (10, 11, 9), c, pos, table=t)
    M = pos.shape[0]
    hpos = torch.from_numpy(pos).pin_memory()
    hval = torch.empty((M, ld), dtype=torch.float32).pin_memory()
    hgrad = torch.empty((M, 3, ld), dtype=torch.float32).pin_memory()
    hlap = torch.empty((M, ld), dtype=torch.float32).pin_memory()
    hcell = torch.empty((M, 3), dtype=torch.int32).pin_memory()
    blip.blipgpu_eval_host(t.handle, hpos, M, blip.VGL, hval, hgrad, hlap, ld, hcell)
    assert np.array_equal(hval.numpy()[:, :L], dev[0])
    assert np.array_equal(hgrad.numpy()[:, :, :L], dev[1])
    assert np.array_equal(hlap.numpy()[:, :L], dev[2])
    assert np.array_equal(hcell.numpy(), dev[3])
    # pageable numpy buffers, value-only
    nval = np.empty((M, ld), dtype=np.float32)
    blip.blipgpu_eval_host(t.handle, pos, M, blip.VALUE, nval, None, None, ld, None)
    assert np.array_equal(nval[:, :L], dev[0])
    t.close()


def test_eval_host_staged_path_large_batch(torch_cuda, blip):
    """blipgpu_eval_host on the staged path with more than 8,192 positions: one evaluation of the
    whole batch, the bits of blipgpu_eval."""
    torch = torch_cuda
    grid, L, M = (17, 12, 19), 257, 20000
    A, c, pos = workloads.small_case(grid, L, M, TRICLINIC, seed=14, spread=3.0)
    ld = 260
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_tuning(t.handle, path=2)
    dev = run_gpu(torch, blip, A, grid, c, pos, table=t)
    hpos = torch.from_numpy(pos).pin_memory()
    hval = torch.empty((M, ld), dtype=torch.float32).pin_memory()
    hgrad = torch.empty((M, 3, ld), dtype=torch.float32).pin_memory()
    hlap = torch.empty((M, ld), dtype=torch.float32).pin_memory()
    n0 = t.launch_count()
    blip.blipgpu_eval_host(t.handle, hpos, M, blip.VGL, hval, hgrad, hlap, ld, None)
    assert t.launch_count() - n0 == 2 and blip.blipgpu_last_path(t.handle) == 2
    assert np.array_equal(hval.numpy()[:, :L], dev[0])
    assert np.array_equal(hgrad.numpy()[:, :, :L], dev[1])
    assert np.array_equal(hlap.numpy()[:, :L], dev[2])
    # grouped direct path, 8,192 < M <= 10,240 (the remainder used to run another kernel)
    blip.blipgpu_set_tuning(t.handle, path=1)
    dev = run_gpu(torch, blip, A, grid, c, pos[:9000], table=t)
    blip.blipgpu_eval_host(t.handle, hpos, 9000, blip.VGL, hval, hgrad, hlap, ld, None)
    assert np.array_equal(hval.numpy()[:9000, :L], dev[0]) and np.array_equal(hlap.numpy()[:9000, :L], dev[2])
    t.close()


@pytest.mark.parametrize("path", [1, 2])
def test_grouped_call_replayed_from_a_cuda_graph(torch_cuda, blip, path):
    """A grouped / staged blipgpu_eval (M > 2,048: bin, scan, scatter, evaluate) keeps no state
    between calls, so it can be captured in a CUDA graph and replayed: three calls (an odd number)
    on two batches are captured once and replayed five times; every replay returns the bits of
    the eager calls, and eager calls after the replays still do."""
    torch = torch_cuda
    grid, L = (17, 12, 19), 257
    A, c, pos = workloads.small_case(grid, L, 9000, TRICLINIC, seed=15, spread=3.0)
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_tuning(t.handle, path=path)
    blip.blipgpu_reserve(t.handle, 9000)
    da, db = torch.from_numpy(pos).cuda(), torch.from_numpy(pos[:5000][::-1].copy()).cuda()
    ld = t.ld

    def bufs(M):
        return (torch.zeros((M, ld), dtype=torch.float32, device="cuda"), torch.zeros((M, 3, ld), dtype=torch.float32, device="cuda"),
                torch.zeros((M, ld), dtype=torch.float32, device="cuda"))

    ref_a, ref_b = bufs(9000), bufs(5000)
    blip.blipgpu_eval(t.handle, da, 9000, blip.VGL, *ref_a, ld)
    blip.blipgpu_eval(t.handle, db, 5000, blip.VGL, *ref_b, ld)
    torch.cuda.synchronize()
    out_a, out_b, out_c = bufs(9000), bufs(5000), bufs(9000)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        blip.blipgpu_eval(t.handle, da, 9000, blip.VGL, *out_a, ld, None, side)
        blip.blipgpu_eval(t.handle, db, 5000, blip.VGL, *out_b, ld, None, side)
        blip.blipgpu_eval(t.handle, da, 9000, blip.VGL, *out_c, ld, None, side)
    for _ in range(5):
        for o in (*out_a, *out_b, *out_c):
            o.zero_()
        graph.replay()
        torch.cuda.synchronize()
        for r, o in zip((*ref_a, *ref_b, *ref_a), (*out_a, *out_b, *out_c)):
            assert torch.equal(r, o)
    again = bufs(9000)
    blip.blipgpu_eval(t.handle, da, 9000, blip.VGL, *again, ld)
    torch.cuda.synchronize()
    for r, o in zip(ref_a, again):
        assert torch.equal(r, o)
    del graph
    t.close()


def test_argument_errors(torch_cuda, blip):
    torch = torch_cuda
    A, c, pos = workloads.small_case((4, 4, 4), 6, 8, SKEW, seed=2)
    t = blip.BlipTable(A, (4, 4, 4), 6, c)
    L = blip.lib()
    dpos = torch.from_numpy(pos).cuda()
    out = torch.empty((8, 8), dtype=torch.float32, device="cuda")
    g = torch.empty((8, 3, 8), dtype=torch.float32, device="cuda")

    def ev(M=8, mode=1, val=out, grad=g, lap=out, ld=8, p=dpos):
        q = lambda x: ctypes.c_void_p(0 if x is None else x.data_ptr())
        return L.blipgpu_eval(t.handle, q(p), M, mode, q(val), q(grad), q(lap), ld, None, None)

    assert ev() == blip.OK
    assert ev(M=-1) == blip.EINVAL
    assert ev(mode=3) == blip.EINVAL
    assert ev(ld=4) == blip.EINVAL            # ld < L
    assert ev(ld=10) == blip.EINVAL           # ld % 4 != 0
    assert ev(val=None) == blip.EINVAL
    assert ev(grad=None) == blip.EINVAL
    assert ev(p=None) == blip.EINVAL
    assert ev(mode=0, grad=None, lap=None) == blip.OK
    mis = out.view(-1)[1:]
    assert L.blipgpu_eval(t.handle, ctypes.c_void_p(dpos.data_ptr()), 1, 0, ctypes.c_void_p(mis.data_ptr()),
                          None, None, 8, None, None) == blip.EINVAL
    torch.cuda.synchronize()
    t.close()


def test_distinct_handles_on_distinct_streams(torch_cuda, blip):
    """include/blipgpu.h: "distinct handles are independent".  Three tables evaluated at the same
    time on three streams (persistent staged kernels competing for the SMs) return the bits of
    their stand-alone evaluation."""
    torch = torch_cuda
    cases = []
    for k, (grid, L, M) in enumerate([((17, 12, 19), 257, 9000), ((9, 10, 13), 130, 30000), ((20, 7, 8), 128, 12000)]):
        A, c, pos = workloads.small_case(grid, L, M, TRICLINIC, seed=k, spread=3.0)
        t = blip.BlipTable(A, grid, L, c)
        blip.blipgpu_set_tuning(t.handle, path=2)
        dpos = torch.from_numpy(pos).cuda()
        ref = [x.clone() for x in t.eval(dpos, mode=blip.VGL)[:3]]
        cases.append((t, dpos, ref, torch.cuda.Stream()))
    torch.cuda.synchronize()
    for _ in range(5):
        outs = []
        for t, dpos, ref, st in cases:
            with torch.cuda.stream(st):
                M, ld = dpos.shape[0], t.ld
                val = torch.empty((M, ld), dtype=torch.float32, device="cuda")
                grad = torch.empty((M, 3, ld), dtype=torch.float32, device="cuda")
                lap = torch.empty((M, ld), dtype=torch.float32, device="cuda")
                blip.blipgpu_eval(t.handle, dpos, M, blip.VGL, val, grad, lap, ld, None, st)
                outs.append((val, grad, lap))
        torch.cuda.synchronize()
        for (t, dpos, ref, st), o in zip(cases, outs):
            L = ref[0].shape[1]
            assert torch.equal(o[0][:, :L], ref[0]) and torch.equal(o[1][:, :, :L], ref[1]) and torch.equal(o[2][:, :L], ref[2])
    for t, *_ in cases:
        t.close()


def test_grouping_with_more_bins_than_fit_in_shared_memory(torch_cuda, blip):
    """A 200^3 grid has 125,000 bricks: the histogram does not fit in the shared memory of the
    one-launch grouping kernel, so the call goes through the three-kernel form (bin, scan,
    scatter); twice, to check that it leaves its histogram clean."""
    grid, L, M = (200, 200, 200), 4, 6000
    lat = ((40.0, 0.0, 0.0), (1.0, 41.0, 0.0), (0.5, 0.25, 39.0))
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=31, spread=1.5)
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_tuning(t.handle, path=1)
    for _ in range(2):
        n0 = t.launch_count()
        out = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
        assert t.launch_count() - n0 == 4 and blip.blipgpu_last_path(t.handle) == 1
        compare(A, grid, c, pos, out)
    t.close()
