"""Recipes for the BASELINE.json configurations C1..C5.

Every array is seeded and synthetic. Arrays are SoA [component][z][y][x], x fastest.
The paper's own benchmark is synthetic as well (uniform Permalloy film, PAPER.md
L1057-L1064); these are stand-ins of the same shape.
"""
import numpy as np
from .rng import uniform01, random_unit_vectors
from .params import Params

SEED0 = 0x14067635


def _random_m(seed, grid):
    nx, ny, nz = grid
    return random_unit_vectors(seed, nx * ny * nz).reshape(3, nz, ny, nx)


def _uniform_m(grid, v):
    nx, ny, nz = grid
    v = np.asarray(v, dtype=np.float64)
    v = v / np.sqrt((v * v).sum())
    m = np.empty((3, nz, ny, nx), dtype=np.float32)
    for c in range(3):
        m[c] = np.float32(v[c])
    return m


def voronoi_regions(seed, grid, ngrains):
    """uint8 region ids [z][y][x]: nearest of `ngrains` seed points uniform in the box.

    Ties go to the lowest seed index. Distances in cell units.
    """
    nx, ny, nz = grid
    g = np.arange(ngrains, dtype=np.uint64)
    px = uniform01(seed, 100, g) * nx
    py = uniform01(seed, 101, g) * ny
    pz = uniform01(seed, 102, g) * nz
    x = np.arange(nx) + 0.5
    y = np.arange(ny) + 0.5
    z = np.arange(nz) + 0.5
    out = np.empty((nz, ny, nx), dtype=np.uint8)
    for iz in range(nz):
        best = np.full((ny, nx), np.inf)
        idx = np.zeros((ny, nx), dtype=np.uint8)
        for k in range(ngrains):
            d = (x[None, :] - px[k]) ** 2 + (y[:, None] - py[k]) ** 2 + (z[iz] - pz[k]) ** 2
            upd = d < best
            best = np.where(upd, d, best)
            idx = np.where(upd, np.uint8(k), idx)
        out[iz] = idx
    return out


def config_c1(grid=(64, 16, 1)):
    """Tiny 2D film, random m, alpha 0.5, B_ext 0; 200 fixed steps of 1e-13 s."""
    return dict(name="C1", grid=grid, cell=(4e-9, 4e-9, 3e-9), pbc=(0, 0, 0), regions=None,
                params=Params.uniform(1, Msat=8.0e5, Aex=1.3e-11, alpha=0.5),
                m0=_random_m(SEED0 + 1, grid), fix_dt=1e-13, nsteps=200)


def config_c2(grid=(128, 32, 1)):
    """Standard-problem-4 geometry 500x125x3 nm."""
    nx, ny, nz = grid
    return dict(name="C2", grid=grid, cell=(500e-9 / nx, 125e-9 / ny, 3e-9), pbc=(0, 0, 0),
                regions=None,
                params=Params.uniform(1, Msat=8.0e5, Aex=1.3e-11, alpha=1.0),
                m0=_uniform_m(grid, (1.0, 0.1, 0.0)), relax_time=5e-9, max_err=1e-5,
                alpha_dyn=0.02, B_ext_dyn=(-24.6e-3, 4.3e-3, 0.0), run_time=1e-9, sample_dt=10e-12)


def config_c3(grid=(128, 128, 32), ngrains=64):
    """3D multi-region block: Voronoi grains, per-region Msat/Ku1/axis, inter-region exchange."""
    seed = SEED0 + 3
    regions = voronoi_regions(seed, grid, ngrains)
    g = np.arange(ngrains, dtype=np.uint64)
    Msat = 6e5 + 4e5 * uniform01(seed, 10, g)
    Ku1 = 5e5 * uniform01(seed, 11, g)
    axes = random_unit_vectors(seed, ngrains, stream=20).astype(np.float64).T.copy()
    ntri = ngrains * (ngrains + 1) // 2
    S = 0.5 + 0.5 * uniform01(seed, 12, np.arange(ntri, dtype=np.uint64))
    for i in range(ngrains):
        S[i * (i + 1) // 2 + i] = 1.0          # S_ii = 1
    p = Params.uniform(ngrains, Msat=Msat, Aex=1.5e-11, alpha=0.1, Ku1=Ku1, exch_scale=S)
    p.anisU = axes
    return dict(name="C3", grid=grid, cell=(2e-9, 2e-9, 2e-9), pbc=(0, 0, 0), regions=regions,
                params=p, m0=_random_m(seed, grid), max_err=1e-5, nsteps=100)


def config_c4(n=4096, seed_offset=0):
    """Large 2D film of the throughput sweep: Permalloy, random m, B_ext 10 mT along x.
    seed_offset selects an independent replica (bench.py --gpus N: one per rank)."""
    grid = (n, n, 1)
    return dict(name="C4-%d" % n, grid=grid, cell=(4e-9, 4e-9, 2e-9), pbc=(0, 0, 0), regions=None,
                params=Params.uniform(1, Msat=8.6e5, Aex=1.3e-11, alpha=0.01, B_ext=(10e-3, 0, 0)),
                m0=_random_m(SEED0 + 4 + 1000 * seed_offset, grid), fix_dt=1e-13, nsteps=1000)


def config_c4_regions(n=4096, ngrains=64):
    """The C4 film cut into `ngrains` Voronoi regions (the structure of C3 in two dimensions): per-region Msat
    within 10 % of Permalloy's, inter-region exchange scaled 0.5-1. Exercises the B_sat gather of the x forward
    kernel and the triangular-table gathers of the stencil at the benchmark size."""
    grid = (n, n, 1)
    seed = SEED0 + 44
    regions = voronoi_regions(seed, grid, ngrains)
    g = np.arange(ngrains, dtype=np.uint64)
    Msat = 8.6e5 * (0.9 + 0.2 * uniform01(seed, 10, g))
    ntri = ngrains * (ngrains + 1) // 2
    S = 0.5 + 0.5 * uniform01(seed, 12, np.arange(ntri, dtype=np.uint64))
    for i in range(ngrains):
        S[i * (i + 1) // 2 + i] = 1.0
    p = Params.uniform(ngrains, Msat=Msat, Aex=1.3e-11, alpha=0.01, B_ext=(10e-3, 0, 0), exch_scale=S)
    return dict(name="C4-%d-regions" % n, grid=grid, cell=(4e-9, 4e-9, 2e-9), pbc=(0, 0, 0), regions=regions,
                params=p, m0=_random_m(SEED0 + 4, grid), fix_dt=1e-13, nsteps=1000)


def config_c5(n=128, pbc=False):
    """Large 3D cube, cubic anisotropy Kc1 = -5e3 J/m^3, optional PBC (4, 4, 0)."""
    grid = (n, n, n)
    return dict(name="C5-%d%s" % (n, "-pbc" if pbc else ""), grid=grid, cell=(2e-9, 2e-9, 2e-9),
                pbc=(4, 4, 0) if pbc else (0, 0, 0), regions=None,
                params=Params.uniform(1, Msat=8.0e5, Aex=1.3e-11, alpha=0.02, Kc1=-5e3),
                m0=_random_m(SEED0 + 5, grid), fix_dt=1e-13, nsteps=100)
