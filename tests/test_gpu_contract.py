"""Parity of blipgpu_eval_contract (evaluation fused with the contraction
of the orbital axis, Eq. 11, 395-399 §VI.D) against the CPU fp64 oracle.

Tolerance: every orbital value may be off by north_star's per-orbital tolerance tol_q, so the
contraction with d_j may be off by tol_q * sum_l |d_j[l]| (max over j of that sum); the fp32
summation over L <= 1,536 terms stays far inside it.
"""
import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import tolerances, torch_cuda, blip  # noqa: F401 (fixtures)

pytestmark = pytest.mark.gpu

TRICLINIC = ((20.0, 0.0, 0.0), (3.0, 19.0, 0.0), (2.0, 2.0, 24.0))


def run_contract(torch, blip, table, pos, d, mode=1, ldd=None, want_cell=False):
    M, L = d.shape
    ldd = (L + 3) // 4 * 4 if ldd is None else ldd
    dd = torch.full((M, ldd), float("nan"), dtype=torch.float32, device="cuda")      # padding must be ignored
    dd[:, :L] = torch.from_numpy(d).cuda()
    out = torch.full((M, 8), 7.0, dtype=torch.float32, device="cuda")
    cell = torch.empty((M, 3), dtype=torch.int32, device="cuda") if want_cell else None
    blip.blipgpu_eval_contract(table.handle, torch.from_numpy(np.ascontiguousarray(pos)).cuda(), M, mode, dd, ldd,
                               out, cell)
    torch.cuda.synchronize()
    return out.cpu().numpy(), None if cell is None else cell.cpu().numpy()


def check(A, grid, c, pos, d, out, mode=1, margin=0.05):
    """Bound: every orbital value may be off by the tolerance, so the contraction by tol x sum_l |d_l|
    (worst case, all errors aligned).  Rounding errors do not align: the measured error must stay
    below `margin` = 5 % of that bound (it sits at ~0.1 % of it), so that a regression of the
    kernel's accuracy by two orders of magnitude fails here, not only one of four."""
    oval, ograd, olap, _ = oracle.eval_fast(A, grid, c, pos, mode=mode)
    ref = oracle.contract(oval, ograd if mode == 1 else None, olap if mode == 1 else None, d)
    tv, tg, tl = tolerances(A, grid, float(np.abs(c).max()))
    w = float(np.abs(d).sum(axis=1).max())
    frac = {"val": float(np.abs(out[:, 0] - ref[:, 0]).max() / (tv * w))}
    if mode == 1:
        frac["grad"] = float(np.abs(out[:, 1:4] - ref[:, 1:4]).max() / (tg * w))
        frac["lap"] = float(np.abs(out[:, 4] - ref[:, 4]).max() / (tl * w))
        assert not out[:, 5:].any()
    else:
        assert not out[:, 1:].any()
    print("contraction error as a fraction of the bound:", {k: round(v, 4) for k, v in frac.items()})
    assert max(frac.values()) < margin, frac
    return frac


@pytest.mark.parametrize("grid,L,M,lat,path", [
    ((9, 10, 13), 130, 3000, TRICLINIC, 2),                # staged kernel, ragged orbital tile
    ((9, 10, 13), 130, 3000, TRICLINIC, 1),                # direct kernel, grouped
    ((6, 5, 7), 37, 300, TRICLINIC, 0),                    # split kernel, L not a multiple of 4
    ((11, 9, 14), 140, 5000, ((7.0, 0, 0), (0, 8.5, 0), (0, 0, 9.25)), 2),   # diagonal-lattice mode
])
def test_contract_small_cases(torch_cuda, blip, grid, L, M, lat, path):
    A, c, pos = workloads.small_case(grid, L, M, lat, seed=L + M, spread=2.5)
    d = np.random.default_rng(M).standard_normal((M, L)).astype(np.float32)
    t = blip.BlipTable(A, grid, L, c)
    blip.blipgpu_set_tuning(t.handle, path=path)
    for mode in (1, 0):
        out, cell = run_contract(torch_cuda, blip, t, pos, d, mode=mode, ldd=(L + 3) // 4 * 4 + 8, want_cell=True)
        assert blip.blipgpu_last_path(t.handle) == (path if path else 3)
        ocell, _ = oracle.cellmap(A, grid, pos)
        assert np.array_equal(cell, ocell)
        check(A, grid, c, pos, d, out, mode=mode)
    t.close()


def test_contract_non_finite_and_empty(torch_cuda, blip):
    grid, L = (8, 8, 8), 12
    A, c, pos = workloads.small_case(grid, L, 64, TRICLINIC, seed=1)
    pos[7, 2] = np.nan
    d = np.ones((64, L), dtype=np.float32)
    t = blip.BlipTable(A, grid, L, c)
    out, _ = run_contract(torch_cuda, blip, t, pos, d)
    assert np.isnan(out[7, :5]).all() and np.isfinite(np.delete(out, 7, axis=0)).all()
    good = np.arange(64) != 7
    check(A, grid, c, pos[good], d[good], out[good])
    n0 = t.launch_count()
    blip.blipgpu_eval_contract(t.handle, None, 0, 1, None, 12, None)       # M = 0: nothing launched
    assert t.launch_count() == n0
    assert blip.lib().blipgpu_eval_contract(t.handle, None, 5, 1, None, 12, None, None, None) == blip.EINVAL
    t.close()


def test_contract_tio2_full_size_every_output(torch_cuda, blip):
    """The bench configuration (staged kernel, 49,152 x 768): every position's five sums."""
    cfg = workloads.CONFIGS["tio2"]
    A = workloads.lattice(cfg)
    c = workloads.coefficients(cfg.grid, cfg.norb)
    pos = workloads.positions(cfg)
    d = workloads.contraction_vectors(pos.shape[0], cfg.norb)
    t = blip.BlipTable(A, cfg.grid, cfg.norb, c)
    out, _ = run_contract(torch_cuda, blip, t, pos, d)
    assert blip.blipgpu_last_path(t.handle) == 2
    t.close()
    tv, tg, tl = tolerances(A, cfg.grid, float(np.abs(c).max()))
    assert not out[:, 5:].any()
    worst = 0.0
    for lo in range(0, pos.shape[0], 8192):
        hi = min(lo + 8192, pos.shape[0])
        oval, ograd, olap, _ = oracle.eval_fast(A, cfg.grid, c, pos[lo:hi])
        ref = oracle.contract_rows(oval, ograd, olap, d[lo:hi])
        w = float(np.abs(d[lo:hi]).sum(axis=1).max())
        worst = max(worst, float(np.abs(out[lo:hi, 0] - ref[:, 0]).max() / (tv * w)),
                    float(np.abs(out[lo:hi, 1:4] - ref[:, 1:4]).max() / (tg * w)),
                    float(np.abs(out[lo:hi, 4] - ref[:, 4]).max() / (tl * w)))
    print("contraction error as a fraction of the worst-case bound, all 49,152 positions:", round(worst, 4))
    assert worst < 0.05, worst                               # see check(): ~0.1 % expected
