"""Pins for the merged acceleration cells of the oracle.

P:54 only says the acceleration grid is "of coarser resolution than the simulation"; any majorant >= k_ext
leaves every expectation unchanged, so merging blocks of cells where the extinction is nearly uniform may
only change the sample paths.  Pinned here against things other than the oracle itself: the table against a
brute-force numpy construction; the traversal (level changes keep the photon where it is) against the exact
direct-beam integrator per landing column; the voxel lookup inside a merged cell against Beer-Lambert
per level; expectations against the single-level run on a cumulus field."""
import numpy as np

import oracle as O
from rt_inputs import CONFIGS, make_optics, plane_parallel
from test_oracle_pins import T, W0, _slant_optical_depth, frac, within


def _brute_table(k, b, m, ratio):
    """-(block max) where max <= ratio * min over the block's voxels (fp32), else the cell's own max."""
    nz, ny, nx = k.shape
    ncz, ncy, ncx = nz // b[2], ny // b[1], nx // b[0]
    cell = k.reshape(ncz, b[2], ncy, b[1], ncx, b[0]).max(axis=(1, 3, 5))
    out = cell.copy()
    if tuple(m) == (1, 1, 1):                              # single-level grid: no sign bits at all
        return out
    sz, sy, sx = m[2] * b[2], m[1] * b[1], m[0] * b[0]
    for Z in range(nz // sz):
        for Y in range(ny // sy):
            for X in range(nx // sx):
                blk = k[Z * sz:(Z + 1) * sz, Y * sy:(Y + 1) * sy, X * sx:(X + 1) * sx]
                hi, lo = np.float32(blk.max()), np.float32(blk.min())
                if hi <= np.float32(ratio) * lo:
                    out[Z * m[2]:(Z + 1) * m[2], Y * m[1]:(Y + 1) * m[1], X * m[0]:(X + 1) * m[0]] = -hi
    return out


def test_merged_table_brute_force():
    rng = np.random.default_rng(11)
    nx, ny, nz = 32, 16, 24
    k = (1e-4 * rng.uniform(1.0, 1.2, size=(nz, ny, nx))).astype(np.float32)
    k[rng.uniform(size=k.shape) < 0.004] = 0.03            # a few cloudy voxels break up some blocks
    k[:4] = 0.0                                            # a vacuum layer merges with sign bit on -0.0
    for b, m, ratio in (((2, 2, 2), (4, 2, 2), 1.25), ((2, 2, 1), (2, 4, 4), 1.1), ((4, 4, 4), (1, 1, 1), 1.25)):
        got = O.majorant(nx, ny, nz, *b, k, merge=m, merge_ratio=ratio)
        want = _brute_table(k, b, m, ratio)
        assert np.array_equal(got.view(np.uint32), want.view(np.uint32)), (b, m)
        if m != (1, 1, 1):
            assert np.signbit(got).any() and not np.signbit(got).all()
            assert np.signbit(got[:2]).all()               # the vacuum layer: -0.0


def _field_with_clear_air(nx, ny, nz, rng):
    """Uniform thin gas with two compact cloudy clusters: most 4x4x2-cell blocks merge, some do not."""
    k = np.full((nz, ny, nx), 2e-4)
    k[6:10, 3:8, 9:14] = rng.uniform(2e-3, 8e-3, size=(4, 5, 5))
    k[3:6, 12:15, 1:4] = rng.uniform(2e-3, 8e-3, size=(3, 3, 3))
    return k


def test_direct_beam_through_merged_cells():
    """Same pin as test_direct_beam_heterogeneous_field, with merged cells: P(unscattered arrival in a
    given column) = exp(-int k_ext ds) along the periodic slant ray from an independent integrator.  A
    level change that moved the photon, lost part of the residual optical depth or picked the wrong cell
    of the entered block would put direct light into the wrong columns or attenuate it wrongly."""
    nx = ny = 16
    nz, dx, dy, dz, zen, azi = 16, 100.0, 100.0, 50.0, 35.0, 250.0
    k = _field_with_clear_air(nx, ny, nz, np.random.default_rng(3))
    cfg, opt = plane_parallel(nx, ny, nz, dx, dy, dz, 0.0, 0.0, albedo=0.3, block=(2, 2, 2))
    opt["k_ext"] = k.astype(np.float32)
    opt["ssa"] = np.full_like(opt["k_ext"], 0.9)
    opt["k_ext_cloud"] = (0.5 * opt["k_ext"]).astype(np.float32)
    opt["g"][:] = 0.6
    n = nx * ny * 2048
    th, ph = np.radians(zen), np.radians(azi)
    sx, sy, sz = -np.sin(th) * np.sin(ph), -np.sin(th) * np.cos(ph), -np.cos(th)
    m = 12
    sub = (np.arange(m) + 0.5) / m
    X0 = ((np.arange(nx)[None, :, None, None] + sub[None, None, None, :]) * dx)
    Y0 = ((np.arange(ny)[:, None, None, None] + sub[None, None, :, None]) * dy)
    X0, Y0 = np.broadcast_arrays(X0, Y0)
    x0, y0 = X0.ravel().astype(np.float64), Y0.ravel().astype(np.float64)
    tau = _slant_optical_depth(opt["k_ext"].astype(np.float64), dx, dy, dz, x0, y0, sx, sy, sz)
    s_end = nz * dz / -sz
    lx = np.floor((x0 + sx * s_end) / dx).astype(np.int64) % nx
    ly = np.floor((y0 + sy * s_end) / dy).astype(np.int64) % ny
    expect = np.zeros((ny, nx))
    np.add.at(expect, (ly, lx), np.exp(-tau) * (n / (nx * ny)) / (m * m))
    for merge in ((2, 2, 2), (4, 4, 2), (2, 4, 4)):
        t, _, _ = O.trace((nx, ny, nz, dx, dy, dz, 2, 2, 2), opt, zen, azi, n, seed=5, n_threads=T, merge=merge)
        assert t.closure() == n * W0
        assert t.counters.n_relevel > n // 2               # photons do pass between the two levels
        got = t.sfc_dir.astype(np.float64) / W0
        chi2 = float((((got - expect) ** 2) / np.maximum(expect, 1.0)).sum())
        dof = nx * ny
        assert chi2 < 1.05 * (dof + 4 * np.sqrt(2 * dof)), (merge, chi2, dof)
        within(got.sum() / n, expect.sum() / n, n, extra=2e-4)


def test_beer_lambert_inside_merged_cells():
    """omega0 = 0 and a per-level profile within the merge ratio: the whole domain is merged cells of
    4 x 4 x 4 acceleration cells (8 levels each).  Absorption per LEVEL must still be the difference of
    exponentials: pins the voxel lookup inside a merged cell (which of its m b voxels per axis) and the
    use of the block maximum as majorant (nulls occur and must not bias anything)."""
    nz, dz, zen = 16, 100.0, 50.0
    kz = 4e-4 * (1.0 + 0.2 * np.sin(np.arange(nz) * 1.7) ** 2)
    cfg, opt = plane_parallel(16, 16, nz, 100.0, 100.0, dz, kz, 0.0, albedo=0.0, block=(2, 2, 2))
    n = 1 << 19
    t, _, _ = O.trace(cfg.grid, opt, zen, 33.0, n, seed=3, n_threads=T, merge=(4, 4, 4), merge_ratio=1.25)
    tab = O.majorant(16, 16, nz, 2, 2, 2, opt["k_ext"], merge=(4, 4, 4), merge_ratio=1.25)
    assert np.signbit(tab).all() and t.counters.n_relevel == 0
    mu0 = np.cos(np.radians(zen))
    k32 = opt["k_ext"][:, 0, 0].astype(np.float64)
    trans = np.exp(-np.concatenate([[0.0], np.cumsum(k32[::-1] * dz)]) / mu0)
    assert t.closure() == n * W0 and int(t.sfc_dif.sum()) == 0 and int(t.toa_up.sum()) == 0
    within(frac(t.sfc_dir, n), trans[-1], n)
    layer = t.atm_abs.sum(axis=(1, 2))[::-1] / (n * W0)
    expect = trans[:-1] - trans[1:]
    chi2 = float(((layer - expect) ** 2 * n / expect).sum())
    assert chi2 < nz + 4 * np.sqrt(2 * nz), chi2
    assert t.counters.n_null > 0
    # columns are exchangeable in a plane-parallel medium also when photons cross merged cells obliquely
    col = t.atm_abs.sum(axis=0).astype(np.float64) / W0
    chi2c = float(((col - col.mean()) ** 2 / col.mean()).sum())
    assert chi2c < 255 + 4 * np.sqrt(2 * 255), chi2c


def test_merged_cells_leave_expectations_unchanged():
    """BASELINE.json configs[1] field (128x128x64 cumulus): with and without merged cells the five
    domain-mean fractions agree within Monte Carlo noise and the surface pattern (16x16-column block sums)
    agrees bin by bin, while the number of cell crossings drops (by 46 % on this shallow domain)."""
    cfg = CONFIGS[2]
    opt = make_optics(cfg)
    n = 1 << 19
    grid = cfg.grid[:6] + (2, 2, 2)
    a, _, _ = O.trace(grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=21, n_threads=T)
    b, _, _ = O.trace(grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=22, n_threads=T, merge=(8, 8, 4))
    assert a.closure() == n * W0 and b.closure() == n * W0
    assert a.counters.n_relevel == 0 and b.counters.n_relevel > n
    assert b.counters.n_cell_steps < 0.7 * a.counters.n_cell_steps
    for name in ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up"):
        pa, pb = frac(getattr(a, name), n), frac(getattr(b, name), n)
        pm = 0.5 * (pa + pb)
        assert abs(pa - pb) < 4 * np.sqrt(2 * pm * (1 - pm) / n), (name, pa, pb)
    sa = (a.sfc_dir + a.sfc_dif).reshape(8, 16, 8, 16).sum(axis=(1, 3)).astype(np.float64) / W0
    sb = (b.sfc_dir + b.sfc_dif).reshape(8, 16, 8, 16).sum(axis=(1, 3)).astype(np.float64) / W0
    chi2 = float(((sa - sb) ** 2 / (sa + sb)).sum())
    assert chi2 < 64 + 4 * np.sqrt(2 * 64), chi2
    ha = a.atm_abs.reshape(8, 8, 8, 16, 8, 16).sum(axis=(1, 3, 5)).astype(np.float64) / W0
    hb = b.atm_abs.reshape(8, 8, 8, 16, 8, 16).sum(axis=(1, 3, 5)).astype(np.float64) / W0
    msk = (ha + hb) >= 50
    chi2h = float(((ha - hb)[msk] ** 2 / (ha + hb)[msk]).sum())
    assert chi2h < msk.sum() + 4 * np.sqrt(2 * msk.sum()), (chi2h, int(msk.sum()))


def test_voxel_sized_cells_have_no_null_collisions_and_the_same_expectations():
    """Acceleration cells of ONE voxel (Q1: the bench configuration of configs 3 and 5), merged 4 x 4 x 4 in
    clear air: the majorant of an unmerged cell is the voxel's own extinction, so a null collision can only happen
    inside a merged cell (n_null <= the events of photons at level 1, here under 1 % of all events), every other
    event is real; and the expectations are those of the 4^3-voxel single-level grid of BASELINE.json configs[1]
    (domain means within 4 sigma, 16 x 16-column surface sums bin by bin)."""
    cfg = CONFIGS[2]
    opt = make_optics(cfg)
    n = 1 << 19
    a, _, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=31, n_threads=T)
    b, _, _ = O.trace(cfg.grid[:6] + (1, 1, 1), opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=32, n_threads=T,
                      merge=(4, 4, 4))
    assert a.closure() == n * W0 and b.closure() == n * W0
    ca, cb = a.counters, b.counters
    assert ca.n_null > 2 * (ca.n_hg + ca.n_rayleigh)           # the coarse grid spends most events on null collisions
    assert cb.n_null < 0.01 * cb.n_events and cb.n_relevel > n
    # the REAL events are the physics: same rate in both (Poisson-like totals of ~8e6)
    ra, rb = ca.n_events - ca.n_null, cb.n_events - cb.n_null
    assert abs(ra - rb) < 0.01 * ra
    for name in ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up"):
        pa, pb = frac(getattr(a, name), n), frac(getattr(b, name), n)
        pm = 0.5 * (pa + pb)
        assert abs(pa - pb) < 4 * np.sqrt(2 * pm * (1 - pm) / n), (name, pa, pb)
    sa = (a.sfc_dir + a.sfc_dif).reshape(8, 16, 8, 16).sum(axis=(1, 3)).astype(np.float64) / W0
    sb = (b.sfc_dir + b.sfc_dif).reshape(8, 16, 8, 16).sum(axis=(1, 3)).astype(np.float64) / W0
    chi2 = float(((sa - sb) ** 2 / (sa + sb)).sum())
    assert chi2 < 64 + 4 * np.sqrt(2 * 64), chi2
