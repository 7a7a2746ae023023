"""Seeded synthetic inputs for the five BASELINE.json configs.

Shared by the oracle tests, the GPU parity tests, smoke() and bench.py.  Holds NONE of the
method's arithmetic (no cell map, no spline weights): it only draws lattices, coefficient
tables and electron positions with the shapes of the paper's workloads — N = 1,536
electrons, 384 complex = 768 real orbitals, a grid of ~50^3-60^3 sites (PAPER.md:82, 108,
120).  The paper's own Si / TiO2 blip wave functions (refs [21], [22]) are not available;
these stand in for them.

Recipe (all numpy PCG64):
  coefficients  N(0,1) fp32, table order [n1][n2][n3][L]; the table is drawn in 16 slabs
                along k1 (np.array_split), slab j from SeedSequence(seed=0).spawn(16)[j],
                so the values do not depend on how many threads draw them;
  positions     u ~ U[0,1)^3 fp64 from default_rng(1 + rank_offset), r = u @ A, delivered
                unsorted, walker-major then electron;
  clustered     (config 3/4) every position with index % 5 == 0 is replaced by site + d,
                site drawn from 96 'atom' sites (uniform in the cell, default_rng(2)), d
                uniform in the 0.5-bohr ball (default_rng(3): direction = normalised
                Gaussian, radius = 0.5 U^(1/3), site index uniform); not re-wrapped.
"""
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np

COEFF_SEED, POS_SEED, SITE_SEED, CLUSTER_SEED = 0, 1, 2, 3
N_SLABS = 16


@dataclass(frozen=True)
class Config:
    name: str
    lattice: tuple            # 3x3 row-major, rows = lattice vectors (bohr)
    grid: tuple               # (n1, n2, n3)
    norb: int                 # L real orbitals
    electrons: int            # per walker
    walkers: int
    clustered: bool = False
    sweep: tuple = field(default=())   # config 4: batch sizes M

    @property
    def M(self):
        return self.electrons * self.walkers

    @property
    def table_bytes(self):
        n = self.grid
        return 4 * n[0] * n[1] * n[2] * self.norb


def _diag(a, b, c):
    return ((a, 0.0, 0.0), (0.0, b, 0.0), (0.0, 0.0, c))


CONFIGS = {
    "tiny": Config("tiny", _diag(10.0, 10.0, 10.0), (16, 16, 16), 32, 64, 1),
    "small": Config("small", _diag(12.0, 12.0, 14.0), (48, 48, 56), 128, 256, 16),
    "tio2": Config("tio2", _diag(17.4, 17.4, 11.2), (64, 64, 40), 768, 1536, 32, clustered=True),
    "sweep": Config("sweep", _diag(17.4, 17.4, 11.2), (64, 64, 40), 768, 1536, 32, clustered=True,
                    sweep=(1, 8, 32, 128, 512, 1536)),
    "large": Config("large", ((20.0, 0.0, 0.0), (3.0, 19.0, 0.0), (2.0, 2.0, 24.0)),
                    (96, 96, 112), 1536, 3072, 8),
}


def lattice(cfg):
    return np.array(cfg.lattice, dtype=np.float64)


def coefficients(grid, norb, seed=COEFF_SEED, out=None, threads=8):
    """fp32 N(0,1) table [n1][n2][n3][L], drawn slab by slab (see module docstring)."""
    n1, n2, n3 = (int(x) for x in grid)
    if out is None:
        out = np.empty((n1, n2, n3, norb), dtype=np.float32)
    assert out.shape == (n1, n2, n3, norb) and out.dtype == np.float32
    seeds = np.random.SeedSequence(seed).spawn(N_SLABS)
    slabs = np.array_split(np.arange(n1), N_SLABS)

    def draw(j):
        ks = slabs[j]
        if len(ks):
            rng = np.random.default_rng(seeds[j])
            rng.standard_normal(dtype=np.float32, out=out[ks[0]:ks[-1] + 1])

    with ThreadPoolExecutor(max_workers=max(1, threads)) as ex:
        list(ex.map(draw, range(N_SLABS)))
    return out


def positions(cfg, M=None, rank=0):
    """Cartesian positions [M][3] fp64 for `cfg` (first M of the full walker-major set).

    rank > 0 draws an independent batch with the same recipe (seeds shifted by 1000*rank);
    bench.py uses it to give every GPU its own walkers under weak scaling.
    """
    A = lattice(cfg)
    total = cfg.M
    off = 1000 * int(rank)
    u = np.random.default_rng(POS_SEED + off).random((total, 3))
    r = u @ A
    if cfg.clustered:
        sites = np.random.default_rng(SITE_SEED).random((96, 3)) @ A
        rng = np.random.default_rng(CLUSTER_SEED + off)
        idx = np.arange(0, total, 5)
        which = rng.integers(0, 96, size=idx.size)
        d = rng.standard_normal((idx.size, 3))
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        rad = 0.5 * rng.random(idx.size) ** (1.0 / 3.0)
        r[idx] = sites[which] + d * rad[:, None]
    if M is not None:
        r = r[:int(M)]
    return np.ascontiguousarray(r)


def small_case(grid, norb, M, lattice_rows, seed=0, spread=3.0):
    """A free-form small case for pins and edge tests: N(0,1) table and positions spread
    over `spread` cells either side of the origin (negative and far-away included)."""
    A = np.array(lattice_rows, dtype=np.float64).reshape(3, 3)
    rng = np.random.default_rng(seed)
    c = rng.standard_normal((*[int(x) for x in grid], norb)).astype(np.float32)
    u = (rng.random((M, 3)) - 0.5) * 2.0 * spread
    return A, c, np.ascontiguousarray(u @ A)


def contraction_vectors(M, norb, seed=4):
    """Per-position vectors d_j [M][norb] fp32 for blipgpu_eval_contract: N(0, 1/norb) entries, the
    scale of a column of the inverse of a well-conditioned norb x norb Slater matrix
    (the paper's matrices are not available)."""
    rng = np.random.default_rng(seed)
    return (rng.standard_normal((int(M), int(norb)), dtype=np.float32) / np.float32(np.sqrt(norb)))


def kpoints(lattice_rows, n_complex, seed=5):
    """Cartesian k-points [n_complex][3] (rad / bohr) for the complex-orbital API: a twist
    q ~ U[-1/2, 1/2)^3 per orbital in units of the reciprocal lattice, k = 2 pi q . (A^-1)^T, i.e.
    anywhere in the first Brillouin zone of the simulation cell (the paper's orbitals are complex,
    PAPER.md:355; its k-points are not given)."""
    A = np.array(lattice_rows, dtype=np.float64).reshape(3, 3)
    q = np.random.default_rng(seed).random((int(n_complex), 3)) - 0.5
    return np.ascontiguousarray(2.0 * np.pi * q @ np.linalg.inv(A).T)
