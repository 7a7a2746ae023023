"""The arithmetic model behind the tensor-core kernel's precision claim (reading R12a),
checked here in numpy, with no GPU and no code of the CUDA path: coefficients and weights are
scaled by a power of two, split in two fp16 terms each (x1 = rn16(x), x2 = rn16(x - x1)), the four
cross products are exact in fp32 and are added in fp32.  The test shows that

* the split carries 22 significant bits: |x - (x1 + x2)| <= max(2^-22 |x|, 2^-25) (the second
  term of a small x is an fp16 subnormal: absolute error 2^-25 on a scale where max |x| is 2^9);
* a 64-term sum built this way stays within 2^-20 sum |c W| of the exact one — a small fraction
  of north_star's tolerances (2e-5 max|c| for values, 5e-5 max|c| / h^2 for Laplacians);
* one fp16 term per operand is NOT enough (it breaks the value tolerance), i.e. the second MMA per
  coefficient term and the [W1 | W2] stacking of the weight tile are needed;
* the scaling keeps tables from 1e-12 to 1e20 and weights up to 1e4 inside the fp16 range;
* the coefficient scale is per orbital: an orbital 1e-6 of the table's maximum keeps the tolerances
  against its own max|c_l|, which a table-wide scale does not.
"""
import numpy as np
import pytest


def split16(x):
    x = np.asarray(x, dtype=np.float32)
    x1 = x.astype(np.float16)
    x2 = (x - x1.astype(np.float32)).astype(np.float16)      # exact difference in fp32, then rounded
    return x1, x2


def pow2_scale(bound, target):
    """2^k with 2^k * bound in (2^(target-1), 2^target]."""
    m, e = np.frexp(np.float64(bound))
    return np.float32(np.ldexp(1.0, target - int(e)))


def tc_sum(c, w, sc, sw, terms=2):
    """sum_s c[s] w[s] the way the MMAs form it (fp16 x fp16 products exact in fp32, fp32 accumulation)."""
    c1, c2 = split16(np.float32(c) * sc)
    w1, w2 = split16(np.float32(w) * sw)
    parts = [(c1, w1)] if terms == 1 else [(c1, w1), (c2, w1), (c1, w2), (c2, w2)]
    acc = np.float32(0.0)
    for a, b in parts:
        for x, y in zip(a.astype(np.float32), b.astype(np.float32)):
            acc = np.float32(acc + np.float32(x * y))         # the product of two fp16 numbers is exact in fp32
    return np.float64(acc) / (np.float64(sc) * np.float64(sw))


def test_two_fp16_terms_carry_22_bits():
    rng = np.random.default_rng(0)
    x = (rng.standard_normal(100000) * 300).astype(np.float32)
    x1, x2 = split16(x)
    err = np.abs(x.astype(np.float64) - (x1.astype(np.float64) + x2.astype(np.float64)))
    assert (err <= np.maximum(2.0 ** -22 * np.abs(x), 2.0 ** -25)).all()
    assert (err > 2.0 ** -26 * np.abs(x)).any()              # and not more than that: fp32 has 24


@pytest.mark.parametrize("cscale", [1e-12, 1.0, 1e20])
@pytest.mark.parametrize("wbound", [1.0, 13.5, 1e4])
def test_site_sum_error_against_the_tolerances(cscale, wbound):
    rng = np.random.default_rng(1)
    worst = 0.0
    for trial in range(200):
        c = (rng.standard_normal(64) * cscale).astype(np.float32)
        w = (rng.uniform(-1, 1, 64) * wbound * rng.uniform(0, 1, 64) ** 3).astype(np.float32)     # many small, a few large
        cmax = np.float32(6.0 * cscale)                      # the table's max |c| (sets the scale), ~6 sigma
        sc, sw = pow2_scale(cmax, 9), pow2_scale(wbound, 8)
        assert np.abs(np.float32(c) * sc).max() <= 512 and np.abs(np.float32(w) * sw).max() <= 256
        exact = float(np.dot(c.astype(np.float64), w.astype(np.float64)))
        got = tc_sum(c, w, sc, sw)
        bound = 2.0 ** -20 * float(np.abs(c.astype(np.float64) * w.astype(np.float64)).sum()) + 1e-30
        assert abs(got - exact) <= bound
        worst = max(worst, abs(got - exact) / (float(cmax) * wbound))
    # value weights sum to 1 (wbound = 1 row): tolerance 2e-5 max|c|; Laplacian weights are bounded by
    # ~12 / h^2 in magnitude sum: tolerance 5e-5 max|c| / h^2 — either way the model is 20 x inside
    assert worst <= 1e-6


def test_per_orbital_scale_keeps_small_orbitals_accurate():
    """The scale is chosen per orbital (2^k_l max|c_l| in [2^8, 2^9)), not per table: an orbital 1e-6 of
    the table's maximum keeps an error of ~2^-21 of ITS sum |c W|.  Under a table-wide scale the same
    orbital sits on the fp16 subnormal floor (absolute error 2^-25 per coefficient on the scaled
    axis) and misses the value tolerance measured against its own max|c_l| by orders of magnitude."""
    rng = np.random.default_rng(3)
    table_max, amp = np.float32(6.0), np.float32(1e-6)
    worst_own, worst_global = 0.0, 0.0
    for trial in range(200):
        c = (rng.standard_normal(64) * amp).astype(np.float32)
        w = rng.dirichlet(np.ones(64)).astype(np.float32)
        own_max = np.float32(6.0) * amp
        exact = float(np.dot(c.astype(np.float64), w.astype(np.float64)))
        sw = pow2_scale(1.0, 8)
        e_own = abs(tc_sum(c, w, pow2_scale(own_max, 9), sw) - exact)
        e_glob = abs(tc_sum(c, w, pow2_scale(table_max, 9), sw) - exact)
        assert e_own <= 2.0 ** -20 * float(np.abs(c.astype(np.float64) * w).sum()) + 1e-36
        worst_own = max(worst_own, e_own / (2e-5 * float(own_max)))
        worst_global = max(worst_global, e_glob / (2e-5 * float(own_max)))
    assert worst_own <= 0.05                                 # 20 x inside the value tolerance against its own max
    assert worst_global > 1.0                                # a table-wide scale breaks it for this orbital


def test_one_fp16_term_is_not_enough():
    rng = np.random.default_rng(2)
    bad = 0
    for trial in range(200):
        c = rng.standard_normal(64).astype(np.float32)
        w = rng.dirichlet(np.ones(64)).astype(np.float32)     # positive weights that sum to 1, like the value weights
        sc, sw = pow2_scale(6.0, 9), pow2_scale(1.0, 8)
        exact = float(np.dot(c.astype(np.float64), w.astype(np.float64)))
        assert abs(tc_sum(c, w, sc, sw) - exact) <= 2e-5 * 6.0 * 0.05
        bad += abs(tc_sum(c, w, sc, sw, terms=1) - exact) > 2e-5 * 6.0 * 0.05
    assert bad > 100                                         # a single term misses what two terms reach in most draws
