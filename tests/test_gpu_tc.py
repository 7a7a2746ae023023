"""The tensor-core form of the staged kernel (blip::eval_tc_kernel, tuning path 5; the kernel the
automatic choice takes for dense batches): parity with the oracle on every output, the cases its
layout makes special (ragged orbital chunks, grids that are not a multiple of the 4 x 4 pencil,
every z offset of an electron in its pencil, non-finite positions, tables of very different
scale), run-to-run bit identity, and the fall-backs."""
import os
import re
import subprocess
import sys

import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import (GRAD_TOL, LAP_TOL, VAL_TOL, compare, compare_all, run_gpu, tolerances,  # noqa: F401 (fixtures)
                             torch_cuda, blip, tio2)

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "tests", "harness"))
import build as harness_build  # noqa: E402


def test_tcgen05_facts_the_kernel_relies_on():
    """tests/harness/tcgen05_check.cu: fp16 pairs per TMEM column (low half first), A operand start at
    multiples of 4 columns, the K-major no-swizzle B descriptor, accumulate flag, fp32 accumulator
    read-back — each against a host loop, for kind::f16 (shipped) and kind::tf32."""
    exe = harness_build.build_tcgen05_check()
    r = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "tcgen05_check: 0 failure(s)" in r.stdout


def test_mma_sync_probe_harness_program_runs():
    """tests/harness/mma_sync_probe.cu — the settled mma.sync tf32 recast experiment,
    moved out of libblipgpu.so: it still builds and times its three forms."""
    exe = harness_build.build_mma_sync_probe()
    r = subprocess.run([exe, "400"], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, r.stdout + r.stderr
    ms = [float(x) for x in re.findall(r"([0-9.]+) ms", r.stdout)]
    assert len(ms) == 3 and all(m > 0 for m in ms), r.stdout


TRICLINIC = ((20.0, 0.0, 0.0), (3.0, 19.0, 0.0), (2.0, 2.0, 24.0))
ORTHO = ((10.0, 0.0, 0.0), (0.0, 9.0, 0.0), (0.0, 0.0, 8.0))


def tc_table(blip, A, grid, c):
    t = blip.BlipTable(A, grid, c.shape[3], c)
    blip.blipgpu_set_tuning(t.handle, path=5)
    return t


@pytest.mark.parametrize("grid,L,lat", [((9, 10, 13), 130, TRICLINIC), ((12, 8, 8), 256, ORTHO), ((7, 5, 6), 128, TRICLINIC),
                                        ((16, 11, 9), 389, ORTHO)])
@pytest.mark.parametrize("mode", [0, 1])
def test_every_output_against_the_oracle(torch_cuda, blip, grid, L, lat, mode):
    """Grids that are not multiples of the pencil (TMA boxes hang over the table edge), orbital
    counts that leave a ragged last chunk, both lattice kinds (kernel MODE 1 and 2), both modes."""
    A, c, pos = workloads.small_case(grid, L, 4000, lat, seed=L + mode, spread=3.0)
    t = tc_table(blip, A, grid, c)
    gpu = run_gpu(torch_cuda, blip, A, grid, c, pos, mode=mode, table=t)
    assert blip.blipgpu_last_path(t.handle) == 5
    compare(A, grid, c, pos, gpu, mode=mode)
    t.close()


@pytest.mark.parametrize("grid,L,M,path", [((45, 8, 8), 128, 6000, 5), ((130, 8, 12), 128, 9000, 5), ((130, 8, 12), 128, 9000, 2),
                                            ((4, 372, 372), 128, 20000, 5)])
def test_segmented_pencils_and_many_work_items(torch_cuda, blip, grid, L, M, path):
    """Pencils cut into segments with a ragged last one (45 planes -> 4 segments of 12, 12, 12, 9), more
    than 4 segments per pencil (the work items are then sorted by load only), and 93 x 93 pencils
    (> 8,192 work items: left in id order, the empty ones skipped by every role of the kernel)."""
    # spacings within 10 % of one another (reading R13a: the Laplacian tolerance is tied to the largest one)
    lat = ((0.26 * grid[0], 0.0, 0.0), (0.4, 0.25 * grid[1], 0.0), (0.1, 0.2, 0.255 * grid[2]))
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=grid[0] + path, spread=1.5)
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_tuning(t.handle, path=path)
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
    assert blip.blipgpu_last_path(t.handle) == path
    pick = np.arange(0, M, 3)
    compare(A, grid, c, pos[pick], (val[pick], grad[pick], lap[pick], cell[pick]))
    t.close()


def test_every_cell_offset_in_a_pencil(torch_cuda, blip):
    """One electron in every cell of an 8 x 8 x 8 grid (all 16 (y0, z0) offsets of a 4 x 4 pencil,
    every plane) plus random ones: the weight tile is placed by z0, the A operand by y0."""
    grid, L = (8, 8, 8), 128
    A, c, _ = workloads.small_case(grid, L, 1, ORTHO, seed=5)
    rng = np.random.default_rng(6)
    cells = np.stack(np.meshgrid(*[np.arange(n) for n in grid], indexing="ij"), -1).reshape(-1, 3)
    u = (cells + rng.random(cells.shape)) / np.asarray(grid)
    pos = np.concatenate([u @ np.asarray(A).reshape(3, 3), rng.random((3000, 3)) @ np.asarray(A).reshape(3, 3)])
    t = tc_table(blip, A, grid, c)
    compare(A, grid, c, pos, run_gpu(torch_cuda, blip, A, grid, c, pos, table=t))
    assert blip.blipgpu_last_path(t.handle) == 5
    t.close()


def test_non_finite_positions_and_far_away_ones(torch_cuda, blip):
    grid, L = (9, 10, 13), 130
    A, c, pos = workloads.small_case(grid, L, 3000, TRICLINIC, seed=9, spread=50.0)
    pos[7] = np.nan
    pos[1234, 1] = np.inf
    t = tc_table(blip, A, grid, c)
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
    assert blip.blipgpu_last_path(t.handle) == 5
    for e in (7, 1234):
        assert np.isnan(val[e]).all() and np.isnan(grad[e]).all() and np.isnan(lap[e]).all() and (cell[e] == -1).all()
    ok = np.ones(len(pos), bool); ok[[7, 1234]] = False
    compare(A, grid, c, pos[ok], (val[ok], grad[ok], lap[ok], cell[ok]))
    t.close()


@pytest.mark.parametrize("scale", [1e-12, 3e-4, 1.0, 7e5, 1e20])
def test_table_scale(torch_cuda, blip, scale):
    """The coefficients go through fp16 after a power-of-two scaling by each orbital's max |c_l|: tables
    far outside the fp16 range keep north_star's tolerances."""
    grid, L = (9, 10, 13), 130
    A, c, pos = workloads.small_case(grid, L, 3000, TRICLINIC, seed=11)
    c = (c * np.float32(scale)).astype(np.float32)
    t = tc_table(blip, A, grid, c)
    compare(A, grid, c, pos, run_gpu(torch_cuda, blip, A, grid, c, pos, table=t))
    assert blip.blipgpu_last_path(t.handle) == 5
    t.close()


@pytest.mark.parametrize("mode", [1, 0])
def test_orbitals_of_very_different_norm_keep_their_own_accuracy(torch_cuda, blip, mode):
    """Real blip tables hold orbitals of very different amplitude (PAPER.md:298-322 relies on
    fp32-accurate orbitals).  The fp16 table is scaled per orbital (the M rows of the MMA are orbitals),
    so every orbital meets north_star's factors against ITS OWN max|c_l| — 2e-5, 2e-5 / h, 5e-5 / h^2 —
    not only against the table's maximum: amplitudes from 1 down to 1e-6 across the 130 orbitals, a
    few all-zero ones, and one orbital 1e-30 of the rest (a table-wide scale would return its fp16
    subnormal floor: relative errors of 1e-2 and worse from 1e-4 down)."""
    grid, L = (9, 10, 13), 130
    A, c, pos = workloads.small_case(grid, L, 3000, TRICLINIC, seed=15)
    amp = (10.0 ** (-6.0 * np.arange(L) / (L - 1))).astype(np.float32)
    rng = np.random.default_rng(16)
    amp = amp[rng.permutation(L)]                           # amplitudes in no particular order along a 128-orbital chunk
    amp[[5, 64, 129]] = 0.0
    amp[100] = 1e-30
    c = (c * amp).astype(np.float32)
    t = tc_table(blip, A, grid, c)
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, grid, c, pos, mode=mode, table=t)
    assert blip.blipgpu_last_path(t.handle) == 5
    oval, ograd, olap, ocell = oracle.eval_fast(A, grid, c, pos, mode=mode)
    assert np.array_equal(cell, ocell)
    cmax_l = np.abs(c).reshape(-1, L).max(axis=0).astype(np.float64)
    h = float(oracle.spacing(A, grid).max())
    worst = {}
    for name, got, want, fac in (("val", val, oval, VAL_TOL), ("grad", grad, ograd, GRAD_TOL / h), ("lap", lap, olap, LAP_TOL / h ** 2)):
        if got is None:
            continue
        err = np.abs(got.astype(np.float64) - want)
        err = err.max(axis=tuple(range(err.ndim - 1)))      # worst over positions (and components), per orbital
        zero = cmax_l == 0
        assert (err[zero] == 0).all(), f"{name}: an all-zero orbital must return exact zeros"
        frac = err[~zero] / (fac * cmax_l[~zero])
        worst[name] = float(frac.max())
        assert frac.max() <= 1.0, f"{name}: orbital {np.flatnonzero(~zero)[frac.argmax()]} is at {frac.max():.2f} of ITS tolerance"
    print("per-orbital worst fraction of tolerance:", worst)
    t.close()


def test_sparse_table_with_a_few_large_entries(torch_cuda, blip):
    """Most coefficients tiny against their orbital's max |c_l| (they fall into fp16's subnormal range
    after scaling): the error bound is absolute in max |c_l|, so the tolerances hold."""
    grid, L = (9, 10, 13), 130
    A, c, pos = workloads.small_case(grid, L, 3000, TRICLINIC, seed=12)
    c = (c * np.float32(1e-6)).astype(np.float32)
    c[::7, ::3, ::5, ::11] = np.float32(3.0)
    t = tc_table(blip, A, grid, c)
    compare(A, grid, c, pos, run_gpu(torch_cuda, blip, A, grid, c, pos, table=t))
    t.close()


def test_non_finite_table_falls_back_to_the_fp32_kernel(torch_cuda, blip):
    """A NaN in the table would reach electrons that do not touch it through the zero-weight rows
    of an MMA: such a table never takes the tensor-core path (EINVAL when forced)."""
    grid, L = (9, 10, 13), 130
    A, c, pos = workloads.small_case(grid, L, 3000, TRICLINIC, seed=13)
    c[4, 5, 6, 77] = np.nan
    t = blip.BlipTable(A, grid, L, c)
    assert blip.lib().blipgpu_set_tuning(t.handle, 5, 0) == blip.EINVAL
    val, grad, lap, cell = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
    assert blip.blipgpu_last_path(t.handle) == 2
    oval, ograd, olap, ocell = oracle.eval_fast(A, grid, c, pos)
    assert np.array_equal(np.isnan(val), np.isnan(oval)) and np.isnan(oval).any() and not np.isnan(oval).all()
    t.close()


def test_contraction_and_complex_entry_points_keep_the_fp32_kernel(torch_cuda, blip):
    torch = torch_cuda
    grid, L = (9, 10, 13), 130
    A, c, pos = workloads.small_case(grid, L, 3000, TRICLINIC, seed=14)
    t = tc_table(blip, A, grid, c)
    M = pos.shape[0]
    d = torch.randn((M, t.ld), dtype=torch.float32, device="cuda")
    out = torch.empty((M, 8), dtype=torch.float32, device="cuda")
    blip.blipgpu_eval_contract(t.handle, torch.from_numpy(pos).cuda(), M, blip.VGL, d, t.ld, out)
    torch.cuda.synchronize()
    assert blip.blipgpu_last_path(t.handle) == 2
    t.close()


def test_tio2_full_size_repeatable_and_close_to_the_fp32_kernel(torch_cuda, blip, tio2):
    """Full TiO2 batch: 20 repeated calls return the bits of the first (no atomics, a fixed MMA
    order per electron: a stale plane, B tile or accumulator would show as a flicker), and the
    results agree with the FP32-pipe staged kernel to a fraction of the tolerances."""
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
        blip.blipgpu_set_tuning(table.handle, path=5)
        first = call()
        assert blip.blipgpu_last_path(table.handle) == 5
        for _ in range(20):
            again = call()
            torch.cuda.synchronize()
            for a, b in zip(first, again):
                assert torch.equal(a, b)
            del again
        blip.blipgpu_set_tuning(table.handle, path=2)
        ref = call()
        torch.cuda.synchronize()
        tv, tg, tl = tolerances(A, cfg.grid, float(np.abs(c).max()))
        assert float((first[0] - ref[0]).abs().max()) < 0.1 * tv
        assert float((first[1] - ref[1]).abs().max()) < 0.1 * tg
        assert float((first[2] - ref[2]).abs().max()) < 0.1 * tl
    finally:
        blip.blipgpu_set_tuning(table.handle, path=0)


def test_replayed_from_a_cuda_graph(torch_cuda, blip):
    """Grouping + tensor-core kernel captured once and replayed (an odd number of times): all state
    between calls lives on the device; the bits of the eager call."""
    torch = torch_cuda
    grid, L = (12, 8, 8), 256
    A, c, pos = workloads.small_case(grid, L, 6000, ORTHO, seed=15)
    t = tc_table(blip, A, grid, c)
    dpos = torch.from_numpy(pos).cuda()
    M, ld = pos.shape[0], t.ld
    val = torch.empty((M, ld), dtype=torch.float32, device="cuda"); grad = torch.empty((M, 3, ld), dtype=torch.float32, device="cuda")
    lap = torch.empty((M, ld), dtype=torch.float32, device="cuda")
    blip.blipgpu_reserve(t.handle, M)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        blip.blipgpu_eval(t.handle, dpos, M, blip.VGL, val, grad, lap, ld, stream=s)
        s.synchronize()
        eager = (val.clone(), grad.clone(), lap.clone())
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            blip.blipgpu_eval(t.handle, dpos, M, blip.VGL, val, grad, lap, ld, stream=s)
        for _ in range(3):
            val.zero_(); grad.zero_(); lap.zero_()
            g.replay()
            s.synchronize()
            assert torch.equal(val, eager[0]) and torch.equal(grad, eager[1]) and torch.equal(lap, eager[2])
    t.close()


def test_soak_random_batch_sizes(torch_cuda, blip, tio2):
    """Thousands of back-to-back calls with random batch sizes and position windows (every tenth the
    full batch, whose checksum must never change): a lost hand-off between the kernel's five roles
    would hang or flicker.  BLIP_SOAK_CALLS (read here) lengthens the run; profiles/r2_checks.md
    records one with 300,000 calls."""
    torch = torch_cuda
    cfg, A, c, table = tio2
    rng = np.random.default_rng(7)
    p = torch.from_numpy(workloads.positions(cfg)).cuda()
    Mmax, ld = p.shape[0], table.ld
    val = torch.empty((Mmax, ld), dtype=torch.float32, device="cuda")
    grad = torch.empty((Mmax, 3, ld), dtype=torch.float32, device="cuda")
    lap = torch.empty((Mmax, ld), dtype=torch.float32, device="cuda")
    ncalls = int(os.environ.get("BLIP_SOAK_CALLS", "5000"))
    ref = None
    try:
        blip.blipgpu_set_tuning(table.handle, path=5)
        for it in range(ncalls):
            M = int(rng.integers(2049, Mmax + 1)) if it % 10 else Mmax
            off = int(rng.integers(0, Mmax - M + 1))
            blip.blipgpu_eval(table.handle, p[off:off + M], M, blip.VGL, val, grad, lap, ld)
            if it % 10 == 0:
                torch.cuda.synchronize()
                s = (float(val[:, :cfg.norb].sum()), float(lap[:, :cfg.norb].abs().max()))
                assert np.isfinite(s[0]) and np.isfinite(s[1])
                ref = s if ref is None else ref
                assert s == ref
        torch.cuda.synchronize()
        assert blip.blipgpu_last_path(table.handle) == 5
    finally:
        blip.blipgpu_set_tuning(table.handle, path=0)


def test_first_dense_call_inside_a_capture_runs_the_fp32_kernel(torch_cuda, blip):
    """The fp16 copy of the table is built on the first dense call; a stream capture cannot allocate,
    so a dense call captured before that (and without blipgpu_reserve) is served by the FP32-pipe
    staged kernel — correct results either way — and the handle then STAYS on that kernel: the kernel
    of a handle's dense batches is decided once, so a later eager call returns the bits the graph
    replay returned.  With blipgpu_reserve ahead of the capture both run the tensor-core kernel."""
    torch = torch_cuda
    grid, L = (12, 8, 8), 256
    A, c, pos = workloads.small_case(grid, L, 6000, ORTHO, seed=16)
    t = blip.BlipTable(A, grid, L, c)
    dpos = torch.from_numpy(pos).cuda()
    M, ld = pos.shape[0], t.ld
    val = torch.empty((M, ld), dtype=torch.float32, device="cuda"); grad = torch.empty((M, 3, ld), dtype=torch.float32, device="cuda")
    lap = torch.empty((M, ld), dtype=torch.float32, device="cuda")
    cell = torch.empty((M, 3), dtype=torch.int32, device="cuda")
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        # the grouping workspace (an allocation too) is sized ahead of the capture by a call forced to
        # the grouped direct kernel, which does not build the table copy
        blip.blipgpu_set_tuning(t.handle, path=1)
        blip.blipgpu_eval(t.handle, dpos, M, blip.VGL, val, grad, lap, ld, stream=s)
        blip.blipgpu_set_tuning(t.handle, path=0)
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            blip.blipgpu_eval(t.handle, dpos, M, blip.VGL, val, grad, lap, ld, cell, stream=s)
        captured_path = blip.blipgpu_last_path(t.handle)
        g.replay()
        s.synchronize()
    assert captured_path == 2
    compare(A, grid, c, pos, (val.cpu().numpy()[:, :L], grad.cpu().numpy()[:, :, :L], lap.cpu().numpy()[:, :L], cell.cpu().numpy()))
    replayed = val.cpu().numpy()[:, :L].copy()
    out = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
    assert blip.blipgpu_last_path(t.handle) == 2            # decided once: still the FP32-pipe kernel
    assert np.array_equal(out[0], replayed)                 # ... hence the same bits as the replay
    compare(A, grid, c, pos, out)
    assert blip.lib().blipgpu_set_tuning(t.handle, 5, 0) == blip.EINVAL
    t.close()
    # the same with blipgpu_reserve before the capture: the tensor-core kernel, captured and eager
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_reserve(t.handle, M)
    with torch.cuda.stream(s):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            blip.blipgpu_eval(t.handle, dpos, M, blip.VGL, val, grad, lap, ld, cell, stream=s)
        assert blip.blipgpu_last_path(t.handle) == 5
        g.replay()
        s.synchronize()
    replayed = val.cpu().numpy()[:, :L].copy()
    out = run_gpu(torch_cuda, blip, A, grid, c, pos, table=t)
    assert blip.blipgpu_last_path(t.handle) == 5 and np.array_equal(out[0], replayed)
    t.close()


def test_outputs_beyond_32_bit_element_offsets(torch_cuda, blip):
    """700,000 positions x 2,048 orbitals: the gradient array has 4.3e9 elements, so the epilogue takes
    its 64-bit addressing (smaller calls use 32-bit element offsets).  2,000 sampled positions, spread
    over the whole batch, against the oracle."""
    torch = torch_cuda
    grid, L, M = (8, 8, 8), 2048, 700000
    A, c, _ = workloads.small_case(grid, L, 1, ORTHO, seed=21)
    rng = np.random.default_rng(22)
    pos = rng.random((M, 3)) @ np.asarray(A).reshape(3, 3)
    t = tc_table(blip, A, grid, c)
    dpos = torch.from_numpy(pos).cuda()
    ld = t.ld
    assert 3 * M * ld >= 2 ** 32
    val = torch.empty((M, ld), dtype=torch.float32, device="cuda")
    grad = torch.empty((M, 3, ld), dtype=torch.float32, device="cuda")
    lap = torch.empty((M, ld), dtype=torch.float32, device="cuda")
    blip.blipgpu_eval(t.handle, dpos, M, blip.VGL, val, grad, lap, ld)
    torch.cuda.synchronize()
    assert blip.blipgpu_last_path(t.handle) == 5
    pick = np.sort(rng.choice(M, size=2000, replace=False))
    pick[-1] = M - 1
    ip = torch.from_numpy(pick).cuda()
    gpu = (val[ip].cpu().numpy(), grad[ip].cpu().numpy(), lap[ip].cpu().numpy(), None)
    del val, grad, lap
    compare(A, grid, c, pos[pick], gpu)
    t.close()


def test_two_tensor_core_handles_on_two_streams_at_once(torch_cuda, blip):
    """Every CTA of the tensor-core kernel allocates all 512 tensor-memory columns of its SM
    (tcgen05.alloc blocks until they are free).  Two handles evaluating on two streams at the same
    time must therefore serialise per SM, not deadlock: its 185 KB of shared memory keep a second CTA
    off the SM until the first has exited and released its columns.  20 rounds of overlapping calls
    (each stream's kernel is launched while the other's may still run), every result bit-identical
    to the same call made alone."""
    torch = torch_cuda
    grid, L, M = (12, 12, 16), 256, 6000
    A1, c1, p1 = workloads.small_case(grid, L, M, TRICLINIC, seed=31)
    A2, c2, p2 = workloads.small_case(grid, L, M, ORTHO, seed=32)
    t1, t2 = tc_table(blip, A1, grid, c1), tc_table(blip, A2, grid, c2)
    try:
        alone = []
        for t, p in ((t1, p1), (t2, p2)):
            val, grad, lap, _ = t.eval(torch.from_numpy(p).cuda(), mode=blip.VGL)
            torch.cuda.synchronize()
            assert blip.blipgpu_last_path(t.handle) == 5
            alone.append((val.clone(), grad.clone(), lap.clone()))
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        d1, d2 = torch.from_numpy(p1).cuda(), torch.from_numpy(p2).cuda()
        outs = [[torch.empty_like(x) for x in alone[0]], [torch.empty_like(x) for x in alone[1]]]
        torch.cuda.synchronize()
        for _ in range(20):
            for t, d, s, o in ((t1, d1, s1, outs[0]), (t2, d2, s2, outs[1])):
                blip.blipgpu_eval(t.handle, d, M, blip.VGL, o[0], o[1], o[2], t.ld, None, s)
        s1.synchronize()
        s2.synchronize()
        for o, a in zip(outs, alone):
            for x, y in zip(o, a):
                assert torch.equal(x[..., :L], y[..., :L])
    finally:
        t1.close()
        t2.close()
