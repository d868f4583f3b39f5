"""The fp64 oracle against an independent brute-force walker (tests/reference_walk.py): global coordinates, no levels,
level-0 cells walked one by one, own Philox and samplers.  Equal photons, record by record, pin what the statistical
pins can only bound: the remaining-distance traversal, the periodic wrap, the collision voxel, and above all the
arithmetic of the changes of level at merged cells, where one rare mis-step would move a photon by one
cell and pass every 4-sigma test."""
import numpy as np
import pytest

import oracle as O
from reference_walk import walk
from rt_inputs import CONFIGS, make_optics

NAMES = ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up")


def _field(nx, ny, nz, seed):
    """Thin gas (exponential in height) with a few dense, noisy boxes: photons scatter tens of times, cross merged
    clear-air blocks in all directions and wrap around the periodic domain."""
    rng = np.random.default_rng(seed)
    z = (np.arange(nz) + 0.5) * 25.0
    k = np.broadcast_to((2.7e-5 * np.exp(-z / 8000.0))[:, None, None], (nz, ny, nx)).copy()
    cloud = np.zeros_like(k)
    for _ in range(10):
        x0, y0, z0 = rng.integers(0, nx - 10), rng.integers(0, ny - 10), rng.integers(2, nz - 8)
        sx, sy, sz = rng.integers(4, 11), rng.integers(4, 11), rng.integers(3, 7)
        cloud[z0:z0 + sz, y0:y0 + sy, x0:x0 + sx] = 0.03 * np.exp(0.6 * rng.standard_normal((sz, sy, sx)))
    kext = k + cloud
    return {"k_ext": kext.astype(np.float32), "k_ext_cloud": cloud.astype(np.float32),
            "ssa": ((0.45 * k + 0.999 * cloud) / kext).astype(np.float32), "g": np.full(k.shape, 0.86, np.float32),
            "sfc_albedo": rng.uniform(0.1, 0.5, size=(ny, nx)).astype(np.float32)}


def _same(grid, opt, zen, azi, n, seed, accel, first=0, stream=0):
    ref_rec, ref_t, ref_c = walk(grid, opt, zen, azi, n, seed=seed, stream_id=stream, first_photon_id=first, **accel)
    t, rec, _ = O.trace(grid, opt, zen, azi, n, seed=seed, stream_id=stream, first_photon_id=first, precision=64,
                        records=True, **accel)
    same = (rec == ref_rec).all(axis=1)
    return same, rec, ref_rec, t, ref_t, ref_c


CASES = [
    # grid (nx, ny, nz, dx, dy, dz, bx, by, bz), merge, zenith, azimuth, photons
    ((32, 32, 16, 50.0, 50.0, 25.0, 2, 2, 2), (1, 1, 1), 40.0, 30.0, 5000),     # single level
    ((32, 32, 16, 50.0, 50.0, 25.0, 2, 2, 2), (4, 4, 2), 60.0, 120.0, 10000),    # merged cells, oblique sun, wraps
    ((32, 32, 16, 50.0, 50.0, 25.0, 2, 2, 1), (2, 4, 4), 25.0, 250.0, 6000),    # anisotropic cells and factors
    ((32, 32, 16, 50.0, 50.0, 25.0, 1, 1, 1), (8, 8, 8), 60.0, 120.0, 10000),    # voxel-sized cells (configs 3, 5)
    ((24, 12, 16, 60.0, 40.0, 25.0, 2, 2, 2), (4, 2, 4), 55.0, 40.0, 6000),     # non-power-of-two cell counts
]


@pytest.mark.parametrize("grid,merge,zen,azi,n", CASES)
def test_oracle_equals_the_brute_force_walker(grid, merge, zen, azi, n):
    nx, ny, nz = grid[:3]
    opt = _field(nx, ny, nz, seed=nx * 7 + merge[0])
    accel = {"merge": merge, "merge_ratio": 1.25}
    n += 37                                               # not a multiple of ncol: a remainder pass
    same, rec, ref_rec, t, ref_t, ref_c = _same(grid, opt, zen, azi, n, 5, accel, first=(1 << 33) + 11, stream=3)
    bad = np.where(~same)[0]
    assert bad.size == 0, (bad[:5], rec[bad[:5]], ref_rec[bad[:5]])
    for name in NAMES:
        assert np.array_equal(getattr(t, name), ref_t[name]), name
    c = t.counters
    for k in ("n_events", "n_null", "n_hg", "n_rayleigh", "n_atm_abs", "n_sfc_hits", "n_sfc_abs", "n_toa"):
        assert getattr(c, k) == ref_c[k], k
    if merge != (1, 1, 1):
        assert c.n_relevel > n // 2                       # the level changes were exercised ...
        assert c.n_cell_steps < ref_c["n_cell_steps"]     # ... and the walker crossed more (level-0) cells for the same photons
    assert c.n_hg > 2 * n and c.n_sfc_hits > 0 and c.n_toa > 0      # a real workout: several scatterings per photon


def test_oracle_equals_the_walker_on_config1():
    cfg = CONFIGS[1]
    opt = make_optics(cfg)
    same, rec, ref_rec, t, ref_t, _ = _same(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, 3000, cfg.seed, {})
    assert same.all()
    for name in NAMES:
        assert np.array_equal(getattr(t, name), ref_t[name]), name
