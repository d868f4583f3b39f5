"""Pins for the oracle's WEIGHTED mode: the paper's own absorption scheme, "Absorption
is handled by using weights ... its weight is reduced at each scattering or null-collision event ... we store
the weight of the incoming ray multiplied with the local absorption probability ... whenever the weight w is
lower than 0.5, we draw a random number rho ... terminated if rho > w, else the weight is set to 1 ... The
local surface albedo is used to reduce the weight after scattering."

Weights are an unbiased estimator of the same radiative transfer solution, so every closed form that pins the
analog tracer pins this mode too; on top: exact integer closure including the roulette ledger, the ledger's
zero mean, identity with the analog run when nothing absorbs, and the variance reduction the paper claims."""
import numpy as np
from scipy import special

import oracle as O
from rt_inputs import CONFIGS, make_optics, plane_parallel
from test_oracle_pins import T, W0, _slant_optical_depth, frac, within


def test_weighted_equals_analog_without_absorption():
    """omega0 = 1 and albedo = 1: no weight is ever lost, xi = c1 + u1 (k_hat - c1) = u1 k_hat, no roulette:
    the weighted run must reproduce the analog run record by record and quantum by quantum."""
    n = 1 << 15
    cfg, opt = plane_parallel(16, 16, 16, 100.0, 100.0, 100.0, 1.5e-3, 1.0, g=0.7, cloud_frac=0.5, albedo=1.0)
    a, ra, _ = O.trace(cfg.grid, opt, 50.0, 80.0, n, seed=2, n_threads=T, records=True)
    w, rw, _ = O.trace(cfg.grid, opt, 50.0, 80.0, n, seed=2, n_threads=T, records=True, weighted=True)
    assert np.array_equal(ra, rw)
    for name in ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up"):
        assert np.array_equal(getattr(a, name), getattr(w, name)), name
    assert w.counters.n_roulette_killed == 0 and w.counters.n_roulette_kept == 0
    assert int(w.toa_up.sum()) == n * W0


def test_weighted_beer_lambert_layered_slab():
    """Same closed form as the analog pin (absorption in level j = difference of exponentials, surface =
    exp(-tau/mu0)), profile varying inside each 8-level cell so that P(absorb) = k/k_hat < 1: weights shrink
    event by event and the roulette runs.  Closure is exact with the ledger; the ledger has zero mean."""
    nz, dz, zen = 16, 100.0, 50.0
    k = 4e-4 * (1.0 + np.sin(np.arange(nz) * 1.7) ** 2)
    cfg, opt = plane_parallel(16, 16, nz, 100.0, 100.0, dz, k, 0.0, albedo=0.0)
    n = 1 << 19
    t, _, _ = O.trace(cfg.grid, opt, zen, 33.0, n, seed=3, n_threads=T, weighted=True)
    c = t.counters
    mu0 = np.cos(np.radians(zen))
    k32 = opt["k_ext"][:, 0, 0].astype(np.float64)
    trans = np.exp(-np.concatenate([[0.0], np.cumsum(k32[::-1] * dz)]) / mu0)
    assert t.closure() == n * W0
    assert int(t.sfc_dif.sum()) == 0 and int(t.toa_up.sum()) == 0
    assert np.array_equal(t.sfc_dir, t.sfc_abs)               # albedo 0: every arriving quantum is absorbed
    within(frac(t.sfc_dir, n), trans[-1], n)
    layer = t.atm_abs.sum(axis=(1, 2))[::-1] / (n * W0)
    expect = trans[:-1] - trans[1:]
    chi2 = float(((layer - expect) ** 2 * n / expect).sum())
    assert chi2 < nz + 4 * np.sqrt(2 * nz), chi2
    assert c.n_roulette_killed > n // 4 and c.n_roulette_kept > n // 100
    # ledger: each roulette changes the energy by a zero-mean amount bounded by W0/2
    net = (c.roulette_lost - c.roulette_gained) / W0
    assert abs(net) < 4 * 0.5 * np.sqrt(c.n_roulette_killed + c.n_roulette_kept), net


def test_weighted_direct_beam_heterogeneous_field():
    """Direct arrivals per landing column: E = exp(-int k_ext ds) (absorption through the weight, scattering
    through the direct flag) from the independent voxel-marching integrator; variance can only be smaller than
    Poisson, so the chi-square bound is one-sided.  Scattering on, albedo 0.3, merged cells on."""
    nx = ny = 16
    nz, dx, dy, dz, zen, azi = 16, 100.0, 100.0, 50.0, 35.0, 250.0
    rng = np.random.default_rng(7)
    k = 2e-4 + 6e-3 * (rng.uniform(size=(nz, ny, nx)) < 0.08) * rng.uniform(0.2, 1.0, size=(nz, ny, nx))
    cfg, opt = plane_parallel(nx, ny, nz, dx, dy, dz, 0.0, 0.0, albedo=0.3, block=(2, 2, 2))
    opt["k_ext"] = k.astype(np.float32)
    opt["ssa"] = np.full_like(opt["k_ext"], 0.6)
    opt["k_ext_cloud"] = (0.5 * opt["k_ext"]).astype(np.float32)
    opt["g"][:] = 0.6
    n = nx * ny * 2048
    t, _, _ = O.trace(cfg.grid, opt, zen, azi, n, seed=5, n_threads=T, weighted=True, merge=(2, 2, 2))
    assert t.closure() == n * W0
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
    got = t.sfc_dir.astype(np.float64) / W0
    chi2 = float((((got - expect) ** 2) / np.maximum(expect, 1.0)).sum())
    dof = nx * ny
    assert chi2 < 1.05 * (dof + 4 * np.sqrt(2 * dof)), (chi2, dof)
    within(got.sum() / n, expect.sum() / n, n, extra=2e-4)


def test_weighted_surface_albedo_and_lambert():
    """Vacuum over albedo 0.22: the reflected weight is floor(W0 a 2^24) / 2^24 per photon up to the roulette,
    so TOD-up / incident = albedo within noise and sfc_abs + toa_up + ledger closes exactly.  Pure absorber over
    albedo 1: TOD-up = exp(-tau/mu0) 2 E3(tau) as in the analog pin (Lambertian pdf 2 mu)."""
    n = 1 << 18
    cfg, opt = plane_parallel(16, 16, 16, 100.0, 100.0, 100.0, 0.0, 0.0, albedo=0.22)
    t, _, _ = O.trace(cfg.grid, opt, 50.0, 80.0, n, seed=4, n_threads=T, weighted=True)
    assert int(t.sfc_dir.sum()) == n * W0 and t.counters.n_events == 0 and t.closure() == n * W0
    a32 = float(np.float32(0.22))
    aq = int(a32 * 2 ** 24)
    assert int(t.sfc_abs.sum()) == n * (W0 - ((W0 * aq) >> 24))      # exact: every photon arrives with W0
    within(frac(t.toa_up, n), a32, n)
    tau, zen, nz, dz = 0.4, 20.0, 8, 250.0
    cfg, opt = plane_parallel(8, 8, nz, 100.0, 100.0, dz, tau / (nz * dz), 0.0, albedo=1.0)
    n = 1 << 19
    t, _, _ = O.trace(cfg.grid, opt, zen, 0.0, n, seed=12, n_threads=T, weighted=True)
    tau32 = float(opt["k_ext"][0, 0, 0]) * nz * dz
    expect = np.exp(-tau32 / np.cos(np.radians(zen))) * 2.0 * special.expn(3, tau32)
    within(frac(t.toa_up, n), expect, n)
    assert int(t.sfc_abs.sum()) == 0 and t.closure() == n * W0


def test_weighted_reduces_heating_noise():
    """weights "accelerate convergence of radiative fluxes and heating rates".  BASELINE.json configs[0]:
    two independent runs per mode; the RMS difference of per-level heating between the two weighted runs is
    well below that of the two analog runs, and the modes agree with each other within the analog noise."""
    cfg = CONFIGS[1]
    opt = make_optics(cfg)
    n = 1 << 17
    runs = {}
    for wt in (False, True):
        for seed in (31, 32):
            t, _, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=seed, n_threads=T, weighted=wt)
            assert t.closure() == n * W0
            runs[(wt, seed)] = t.atm_abs.sum(axis=(1, 2)).astype(np.float64) / (n * W0)
    d_analog = np.sqrt(np.mean((runs[(False, 31)] - runs[(False, 32)]) ** 2))
    d_weight = np.sqrt(np.mean((runs[(True, 31)] - runs[(True, 32)]) ** 2))
    assert d_weight < 0.6 * d_analog, (d_weight, d_analog)
    mean_a = 0.5 * (runs[(False, 31)] + runs[(False, 32)])
    mean_w = 0.5 * (runs[(True, 31)] + runs[(True, 32)])
    assert np.sqrt(np.mean((mean_a - mean_w) ** 2)) < 3 * d_analog


def test_direct_part_of_heating():
    """P:82 reports heating by direct and by diffuse radiation separately.  The optional tally of heating by
    never-scattered photons has a closed form in a homogeneous scattering slab: level j absorbs
    (1 - omega0) (T_{j-1} - T_j) of the incident power directly, T = exp(-k_ext s) along the slant beam
    (extinction removes photons from the direct beam, a share 1 - omega0 of each removal is absorption).
    Both absorption modes; pure absorber: direct = total exactly; fully diffuse source: no direct heating."""
    nz, dz, zen, k, w0 = 16, 100.0, 40.0, 1.1e-3, 0.55
    cfg, opt = plane_parallel(8, 8, nz, 100.0, 100.0, dz, k, w0, g=0.5, cloud_frac=0.6, albedo=0.3)
    n = 1 << 19
    mu0 = np.cos(np.radians(zen))
    k32, w32 = float(opt["k_ext"][0, 0, 0]), float(opt["ssa"][0, 0, 0])
    trans = np.exp(-k32 * dz * np.arange(nz + 1) / mu0)
    expect = (1 - w32) * (trans[:-1] - trans[1:])                       # top level first
    for wt in (False, True):
        t, _, _ = O.trace(cfg.grid, opt, zen, 100.0, n, seed=9, n_threads=T, weighted=wt, heating_split=True)
        assert t.closure() == n * W0
        assert (t.atm_abs_direct <= t.atm_abs).all() and 0 < int(t.atm_abs_direct.sum()) < int(t.atm_abs.sum())
        layer = t.atm_abs_direct.sum(axis=(1, 2))[::-1] / (n * W0)
        chi2 = float(((layer - expect) ** 2 * n / expect).sum())
        assert chi2 < nz + 4 * np.sqrt(2 * nz), (wt, chi2)
        d, _, _ = O.trace(cfg.grid, opt, zen, 100.0, 1 << 14, seed=9, n_threads=T, weighted=wt, heating_split=True,
                          diffuse_fraction=1.0)
        assert int(d.atm_abs_direct.sum()) == 0 and int(d.atm_abs.sum()) > 0
    cfg, opt = plane_parallel(8, 8, nz, 100.0, 100.0, dz, k, 0.0, albedo=0.0)
    t, _, _ = O.trace(cfg.grid, opt, zen, 100.0, 1 << 15, seed=9, n_threads=T, heating_split=True)
    assert np.array_equal(t.atm_abs_direct, t.atm_abs)
