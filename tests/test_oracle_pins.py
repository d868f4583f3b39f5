"""Pins for the fp64 oracle (oracle/rt_oracle.cpp) against what the paper and the mathematics fix.

Nothing here compares the oracle with itself or with the CUDA path.  Each test states the closed
form, invariant or brute-force computation it checks and the passage (PAPER.md line P:n, SURVEY.md
§8(c)) it pins.  All runs are seeded, so the 4-sigma statistical bounds either hold
or fail deterministically."""
import numpy as np
import pytest
from scipy import special

import oracle as O
from rt_inputs import CONFIGS, make_optics, plane_parallel

W0 = O.W0
T = 8  # oracle threads (integer tallies: the result does not depend on it)


def frac(x, n):
    return float(np.asarray(x, dtype=np.float64).sum()) / (n * W0)


def within(p_obs, p_exp, n, k=4.0, extra=0.0):
    sigma = np.sqrt(max(p_exp * (1.0 - p_exp), 1e-300) / n)
    assert abs(p_obs - p_exp) <= k * sigma + extra, (p_obs, p_exp, sigma)


# ------------------------------------------------------------------------------------------------
# Samplers ("Rayleigh phase function ... Henyey-Greenstein phase function")
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("g", [0.85, 0.86, 0.3, -0.4, 5e-4, 0.0])
def test_hg_inverse_cdf(g):
    """CDF_HG(mu) = (1-g^2)/(2g) [ (1+g^2-2 g mu)^(-1/2) - 1/(1+g) ]; the sampler must return the mu
    with CDF(mu) = u (mu increasing in u, mu = +1 is forward), and E[mu] = g."""
    u = (np.arange(200001) + 0.5) / 200001
    mu = O.sample_hg(g, u)
    assert np.all(np.diff(mu) >= 0) and mu.min() >= -1 and mu.max() <= 1
    if abs(g) >= 1e-3:
        cdf = (1 - g * g) / (2 * g) * ((1 + g * g - 2 * g * mu) ** -0.5 - 1 / (1 + g))
    else:
        cdf = (mu + 1) / 2          # isotropic limit; the HG CDF differs from it by O(g) <= 1e-3
    assert np.abs(cdf - u).max() < (1e-12 if abs(g) >= 1e-3 else 1e-3)
    assert abs(mu.mean() - g) < 2e-5 + (1e-3 if 0 < abs(g) < 1e-3 else 0)


def test_rayleigh_inverse_cdf():
    """p(mu) = 3/8 (1 + mu^2): CDF = (mu^3 + 3 mu + 4)/8; E[mu] = 0, E[mu^2] = 2/5."""
    u = (np.arange(200001) + 0.5) / 200001
    mu = O.sample_rayleigh(u)
    assert np.abs((mu ** 3 + 3 * mu + 4) / 8 - u).max() < 1e-12
    assert abs(mu.mean()) < 1e-9 and abs((mu ** 2).mean() - 0.4) < 1e-6
    # end points of the 24-bit lattice
    assert O.sample_rayleigh(np.array([0.0]))[0] == -1.0
    assert abs(O.sample_rayleigh(np.array([1 - 2.0 ** -24]))[0] - 1.0) < 1e-6


def test_hg_sine_keeps_relative_accuracy_at_the_forward_peak():
    """DESIGN.md §3.9 computes 1 - mu and 1 + mu without cancellation and sin(theta) as the root of their product.
    Pin: against the textbook inverse CDF evaluated with 60-digit arithmetic, the fp64 AND the fp32 sampler give
    sin(theta) to a few ulp RELATIVE even where mu is within 1e-7 of 1 (sqrt(1 - mu^2) from a rounded fp32 mu
    would be off by 100 % there), and mu^2 + sin^2 = 1."""
    from mpmath import mp, mpf, sqrt as msqrt
    mp.dps = 60
    for g in (0.86, 0.85, 0.3, -0.4, 1e-4, 0.0):
        us = [k / 2.0 ** 24 for k in (0, 1, 5, 1 << 12, 1 << 23, (1 << 24) - (1 << 10), (1 << 24) - 37, (1 << 24) - 1)]
        mu64, s64 = O.sample_hg(g, np.array(us), with_sine=True)
        mu32, s32 = O.sample_hg(float(np.float32(g)), np.array(us), precision=32, with_sine=True)
        for j, u in enumerate(us):
            for gg, mus, ss, eps in ((g, mu64, s64, 1e-14), (float(np.float32(g)), mu32, s32, 1e-6)):
                G, U = mpf(gg), mpf(u)
                if gg == 0.0:
                    mu_x = 2 * U - 1
                else:
                    q = (1 - G * G) / (1 - G + 2 * G * U)
                    mu_x = (1 + G * G - q * q) / (2 * G)
                s_x = msqrt(max(mpf(0), 1 - mu_x * mu_x))
                assert abs(mpf(float(mus[j])) - mu_x) <= eps, (gg, u)
                assert abs(mpf(float(ss[j])) - s_x) <= eps * s_x * 4 + mpf(10) ** -30, (gg, u, float(ss[j]), float(s_x))
        assert np.abs(mu64 ** 2 + s64 ** 2 - 1).max() < 1e-14


def test_rotation_geometry():
    """New direction d' is a unit vector with d . d' = mu; azimuth 2 pi u turns d' around d through a
    full circle (the perpendicular parts at u and u + 1/2 are opposite, at u + 1/4 orthogonal).  The frame is built
    from a^2 + b^2, so the same tolerance holds 1e-4 rad from the pole as anywhere else; only
    within 1e-6 rad (a^2 + b^2 <= 1e-12) is the direction taken as exactly +-z."""
    rng = np.random.default_rng(11)
    for it in range(400):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        if it % 6 == 0:
            sc = 10.0 ** rng.uniform(-5.5, -2)
            d = np.array([sc * rng.normal(), sc * rng.normal(), rng.choice([-1.0, 1.0])])
            d /= np.linalg.norm(d)          # near a pole, still on the regular branch
        mu, u = rng.uniform(-1, 1), rng.uniform(0, 0.5)
        a = O.rotate(d, mu, u)
        b = O.rotate(d, mu, u + 0.5)
        c = O.rotate(d, mu, u + 0.25)
        assert d[0] ** 2 + d[1] ** 2 > 1e-12
        for v in (a, b, c):
            assert abs(np.linalg.norm(v) - 1) < 1e-12 and abs(v @ d - mu) <= 1e-9
        pa, pb, pc = a - mu * d, b - mu * d, c - mu * d
        assert np.abs(pa + pb).max() < 1e-7 and abs(pa @ pc) < 1e-7
    # the pole branch: d = +-z exactly (and within 1e-6 rad of it): d' = (s cos, s sin, +-mu)
    for sign in (1.0, -1.0):
        for eps in (0.0, 3e-7):
            v = O.rotate([eps, -eps, sign], 0.3, 0.125)
            s = np.sqrt(1 - 0.09)
            assert np.abs(v - np.array([s * np.cos(np.pi / 4), s * np.sin(np.pi / 4), sign * 0.3])).max() < 2e-6
    # the first-order renormalisation 3/2 - n2/2 keeps the norm at 1 over a long chain of scatters, in fp32 too
    for prec, tol in ((64, 1e-13), (32, 4e-7)):
        d = np.array([0.6, 0.0, -0.8])
        for j in range(2000):
            d = O.rotate(d, float(np.cos(0.3 + 0.001 * j)), (0.61803398875 * j) % 1.0, precision=prec,
                         sn=float(np.sin(0.3 + 0.001 * j)))
        assert abs(np.linalg.norm(d) - 1) < tol


# ------------------------------------------------------------------------------------------------
# Free path + null-collision tracking: Beer-Lambert
# ------------------------------------------------------------------------------------------------
def test_beer_lambert_layered_slab():
    """omega0 = 0, albedo = 0, per-level k: surface direct = exp(-tau/mu0); absorption in level j =
    exp(-tau_above_j/mu0) - exp(-tau_above_{j-1}/mu0); no diffuse light and no TOD flux at all.  The
    profile varies inside each 8-level acceleration cell, so nulls occur and must not bias anything."""
    nz, dz, zen = 16, 100.0, 50.0
    k = 4e-4 * (1.0 + np.sin(np.arange(nz) * 1.7) ** 2)
    cfg, opt = plane_parallel(16, 16, nz, 100.0, 100.0, dz, k, 0.0, albedo=0.0)
    n = 1 << 19
    t, _, _ = O.trace(cfg.grid, opt, zen, 33.0, n, seed=3, n_threads=T)
    mu0 = np.cos(np.radians(zen))
    k32 = opt["k_ext"][:, 0, 0].astype(np.float64)
    tau_above = np.concatenate([[0.0], np.cumsum(k32[::-1] * dz)])       # from the top down
    trans = np.exp(-tau_above / mu0)
    assert t.closure() == n * W0
    assert int(t.sfc_dif.sum()) == 0 and int(t.toa_up.sum()) == 0
    assert np.array_equal(t.sfc_dir, t.sfc_abs)
    within(frac(t.sfc_dir, n), trans[-1], n)
    layer = t.atm_abs.sum(axis=(1, 2))[::-1] / (n * W0)                  # top level first
    expect = trans[:-1] - trans[1:]
    chi2 = float(((layer - expect) ** 2 * n / expect).sum())
    assert chi2 < nz + 4 * np.sqrt(2 * nz), chi2
    assert t.counters.n_null > 0 and t.counters.n_rayleigh == 0 and t.counters.n_hg == 0


def _slant_optical_depth(k, dx, dy, dz, x0, y0, sx, sy, sz):
    """Exact integral of k along rays from (x0, y0, top) down direction (sx, sy, sz<0) to z = 0 through
    the periodic voxel grid: all plane crossings sorted, k taken at the midpoint of each segment."""
    nz, ny, nx = k.shape
    top = nz * dz
    s_end = top / -sz
    cuts = [np.zeros_like(x0)[:, None], np.full_like(x0, s_end)[:, None]]
    cuts.append(np.broadcast_to(((top - np.arange(1, nz) * dz) / -sz)[None, :], (x0.size, nz - 1)))
    for p0, sd, d in ((x0, sx, dx), (y0, sy, dy)):
        if abs(sd) < 1e-12:
            continue
        span = abs(sd) * s_end
        m = int(np.ceil(span / d)) + 1
        j = np.arange(1, m + 1)[None, :]
        if sd > 0:
            planes = (np.floor(p0 / d)[:, None] + j) * d
        else:
            planes = (np.ceil(p0 / d)[:, None] - j) * d
        s = (planes - p0[:, None]) / sd
        cuts.append(np.clip(s, 0.0, s_end))
    s = np.sort(np.concatenate(cuts, axis=1), axis=1)
    mid, seg = 0.5 * (s[:, 1:] + s[:, :-1]), np.diff(s, axis=1)
    ix = np.floor((x0[:, None] + sx * mid) / dx).astype(np.int64) % nx
    iy = np.floor((y0[:, None] + sy * mid) / dy).astype(np.int64) % ny
    iz = np.clip(np.floor((top + sz * mid) / dz).astype(np.int64), 0, nz - 1)
    return (k[iz, iy, ix] * seg).sum(axis=1)


def test_direct_beam_heterogeneous_field():
    """P(photon reaches the surface unscattered) = exp(-int k_ext ds) along the periodic slant ray,
    whatever omega0 and the majorant are (SURVEY.md §8(c) "heterogeneous direct beam").  Scattering is
    ON here; the expectation comes from an independent voxel-marching integrator over a lattice of
    entry points.  The landing column is where the straight ray lands, which also pins the azimuth
    convention (azimuth clockwise from north, photons travel away from the sun) and the wrap."""
    nx = ny = 16
    nz, dx, dy, dz, zen, azi = 16, 100.0, 100.0, 50.0, 35.0, 250.0
    rng = np.random.default_rng(7)
    k = 2e-4 + 6e-3 * (rng.uniform(size=(nz, ny, nx)) < 0.08) * rng.uniform(0.2, 1.0, size=(nz, ny, nx))
    cfg, opt = plane_parallel(nx, ny, nz, dx, dy, dz, 0.0, 0.0, albedo=0.3, block=(4, 4, 4))
    opt["k_ext"] = k.astype(np.float32)
    opt["ssa"] = np.full_like(opt["k_ext"], 0.9)
    opt["k_ext_cloud"] = (0.5 * opt["k_ext"]).astype(np.float32)
    opt["g"][:] = 0.6
    n = nx * ny * 2048
    t, _, _ = O.trace((nx, ny, nz, dx, dy, dz, 4, 4, 4), opt, zen, azi, n, seed=5, n_threads=T)
    assert t.closure() == n * W0
    th, ph = np.radians(zen), np.radians(azi)
    sx, sy, sz = -np.sin(th) * np.sin(ph), -np.sin(th) * np.cos(ph), -np.cos(th)
    m = 12                                                  # m x m entry points per column (midpoint rule)
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
    # per landing column: Poisson-like counts around `expect`; plus the total
    chi2 = float((((got - expect) ** 2) / np.maximum(expect, 1.0)).sum())
    dof = nx * ny
    assert chi2 < 1.05 * (dof + 4 * np.sqrt(2 * dof)), (chi2, dof)
    within(got.sum() / n, expect.sum() / n, n, extra=2e-4)
    assert got.sum() / n < 0.95 * np.exp(-opt["k_ext"].astype(np.float64).min() * s_end)  # the field does attenuate


def test_event_counter_poisson_rate():
    """Tentative collisions are a Poisson process of rate khat along the path (P:54 null-collision on
    the acceleration grid), so E[n_events] = khat * E[path length].  Pure absorber with levels
    alternating k_lo, k_hi and 2-level cells: khat = k_hi everywhere and E[L] = sum over levels of
    S_j (1 - exp(-k_j l))/k_j in closed form.  Pins the metric's event counter (null + real)."""
    nz, dz, zen = 16, 100.0, 40.0
    k_lo, k_hi = 3e-4, 1.2e-3
    k = np.where(np.arange(nz) % 2 == 0, k_lo, k_hi)
    cfg, opt = plane_parallel(8, 8, nz, 100.0, 100.0, dz, k, 0.0, albedo=0.0, block=(4, 4, 2))
    n = 1 << 18
    t, _, _ = O.trace((8, 8, nz, 100.0, 100.0, dz, 4, 4, 2), opt, zen, 10.0, n, seed=8, n_threads=T)
    mu0 = np.cos(np.radians(zen))
    l = dz / mu0
    surv, EL = 1.0, 0.0
    for kj in opt["k_ext"][::-1, 0, 0].astype(np.float64):
        EL += surv * (1 - np.exp(-kj * l)) / kj
        surv *= np.exp(-kj * l)
    kh = float(opt["k_ext"].max())
    exp_events = kh * EL
    got = t.counters.n_events / n
    # per-photon event count has variance <= mean + mean^2 (geometric-like tail); use that bound
    sigma = np.sqrt((exp_events + exp_events ** 2) / n)
    assert abs(got - exp_events) < 4 * sigma, (got, exp_events, sigma)
    assert t.counters.n_events == t.counters.n_null + t.counters.n_atm_abs
    # real events alone: every absorbed photon had exactly one
    within(t.counters.n_atm_abs / n, 1 - surv, n)


def test_majorant_block_size_invariance():
    """Expectations do not depend on the acceleration grid (it only accelerates): the same cloudy
    field traced with 2^3, 4^3 and 8^3-voxel cells gives the same domain-mean fractions within MC noise,
    while the event counts differ (more nulls on coarser cells)."""
    cfg = CONFIGS[1]
    opt = make_optics(cfg)
    n = 1 << 17
    res = {}
    for b in (2, 4, 8):
        grid = cfg.grid[:6] + (b, b, b)
        t, _, _ = O.trace(grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=b, n_threads=T)
        assert t.closure() == n * W0
        res[b] = t
    for name in ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up"):
        p = [frac(getattr(res[b], name), n) for b in (2, 4, 8)]
        pm = float(np.mean(p))
        for x in p:
            sigma = np.sqrt(pm * (1 - pm) / n)
            assert abs(x - pm) < 4 * sigma * np.sqrt(2), (name, p)
    # the cube (voxels 12..19) is aligned with 2- and 4-voxel cells: no nulls there, many with 8-voxel cells
    assert res[2].counters.n_null == 0 and res[4].counters.n_null == 0 and res[8].counters.n_null > n
    assert res[2].counters.n_cell_steps > res[4].counters.n_cell_steps > res[8].counters.n_cell_steps


# ------------------------------------------------------------------------------------------------
# Energy, limits, symmetry (SURVEY.md §8(c) pins)
# ------------------------------------------------------------------------------------------------
def test_closure_and_limits():
    n = 1 << 16
    # omega0 = 1 everywhere: nothing is absorbed in the atmosphere, exactly
    cfg, opt = plane_parallel(16, 16, 16, 100.0, 100.0, 100.0, 1.5e-3, 1.0, g=0.7, cloud_frac=0.5, albedo=0.3)
    t, _, _ = O.trace(cfg.grid, opt, 50.0, 80.0, n, seed=2, n_threads=T)
    assert int(t.atm_abs.sum()) == 0 and t.closure() == n * W0
    assert int(t.sfc_abs.sum()) + int(t.toa_up.sum()) == n * W0
    # ... and albedo = 1 as well: everything leaves through the top, exactly
    opt["sfc_albedo"][:] = 1.0
    t, _, _ = O.trace(cfg.grid, opt, 50.0, 80.0, n, seed=2, n_threads=T)
    assert int(t.toa_up.sum()) == n * W0 and int(t.sfc_abs.sum()) == 0
    # vacuum: every photon arrives direct; reflected fraction = albedo (P:56 Lambertian, local albedo)
    cfg, opt = plane_parallel(16, 16, 16, 100.0, 100.0, 100.0, 0.0, 0.0, albedo=0.22)
    t, _, _ = O.trace(cfg.grid, opt, 50.0, 80.0, n, seed=4, n_threads=T)
    assert int(t.sfc_dir.sum()) == n * W0 and int(t.sfc_dif.sum()) == 0 and t.counters.n_events == 0
    within(frac(t.toa_up, n), float(np.float32(0.22)), n)
    assert t.closure() == n * W0
    # per-column albedo is local: columns with albedo 0 reflect nothing, columns with 1 absorb nothing
    opt["sfc_albedo"][:] = 0.0
    opt["sfc_albedo"][:, 8:] = 1.0
    t, _, _ = O.trace(cfg.grid, opt, 0.0, 0.0, n, seed=4, n_threads=T)
    assert int(t.sfc_abs[:, 8:].sum()) == 0 and np.array_equal(t.sfc_abs[:, :8], t.sfc_dir[:, :8])


def test_plane_parallel_columns_exchangeable():
    """Horizontally uniform optics: per-column tallies are exchangeable, chi^2 of column counts against
    their mean ~ ncol - 1 (also exercises the periodic wrap: the slant path crosses the domain ~3 times)."""
    nx = ny = 16
    cfg, opt = plane_parallel(nx, ny, 16, 50.0, 50.0, 100.0, 1.2e-3, 0.95, g=0.8, cloud_frac=0.7, albedo=0.3)
    n = nx * ny * 1024
    t, _, _ = O.trace(cfg.grid, opt, 65.0, 200.0, n, seed=6, n_threads=T)
    assert t.closure() == n * W0
    dof = nx * ny - 1
    for name in ("sfc_dir", "sfc_dif", "sfc_abs", "toa_up"):
        c = getattr(t, name).astype(np.float64) / W0
        chi2 = float(((c - c.mean()) ** 2 / c.mean()).sum())
        # sfc_dir is stratified by launch column (one photon per column per pass), hence under-dispersed
        assert chi2 < dof + 4 * np.sqrt(2 * dof), (name, chi2)
        if name != "sfc_dir":
            assert chi2 > dof - 4 * np.sqrt(2 * dof), (name, chi2)
    a = t.atm_abs.sum(axis=0).astype(np.float64) / W0
    chi2 = float(((a - a.mean()) ** 2 / a.mean()).sum())
    assert abs(chi2 - dof) < 4 * np.sqrt(2 * dof), chi2


# ------------------------------------------------------------------------------------------------
# Surface ("Lambertian"; reading Q6: pdf(mu) = 2 mu) and scattering geometry
# ------------------------------------------------------------------------------------------------
def test_lambertian_reflection_through_absorbing_slab():
    """Pure absorber of vertical optical depth tau over a surface of albedo 1: a reflected photon escapes
    with probability int_0^1 2 mu exp(-tau/mu) dmu = 2 E3(tau), so TOD-up / incident =
    exp(-tau/mu0) * 2 E3(tau).  (Sampling mu uniformly instead would give E2(tau): 0.443 vs 0.574 here.)"""
    tau, zen = 0.4, 20.0
    nz, dz = 8, 250.0
    cfg, opt = plane_parallel(8, 8, nz, 100.0, 100.0, dz, tau / (nz * dz), 0.0, albedo=1.0)
    n = 1 << 19
    t, _, _ = O.trace(cfg.grid, opt, zen, 0.0, n, seed=12, n_threads=T)
    tau32 = float(opt["k_ext"][0, 0, 0]) * nz * dz
    expect = np.exp(-tau32 / np.cos(np.radians(zen))) * 2.0 * special.expn(3, tau32)
    assert abs(2 * special.expn(3, tau32) - special.expn(2, tau32)) > 0.1
    within(frac(t.toa_up, n), expect, n)
    assert int(t.sfc_dif.sum()) == 0 and int(t.sfc_abs.sum()) == 0 and t.closure() == n * W0


def _single_scatter_quadrature(phase, tau, zen_deg, azi_deg):
    """First-order reflected and diffusely transmitted fractions of a homogeneous conservative slab:
    int_0^tau dt/mu0 e^(-t/mu0) int p(cos Theta)/(4 pi) e^(-t/mu) dOmega over the upward hemisphere, and
    the same with e^(-(tau-t)/|mu|) over the downward one.  Midpoint rule in (t, mu, phi)."""
    th, ph = np.radians(zen_deg), np.radians(azi_deg)
    din = np.array([-np.sin(th) * np.sin(ph), -np.sin(th) * np.cos(ph), -np.cos(th)])
    mu0 = np.cos(th)
    nt, nm, nphi = 48, 600, 192
    tt = (np.arange(nt) + 0.5) / nt * tau
    mu = (np.arange(nm) + 0.5) / nm                      # |mu| of the outgoing direction
    phi = (np.arange(nphi) + 0.5) / nphi * 2 * np.pi
    sin = np.sqrt(1 - mu ** 2)
    out = {}
    for sign, name in ((+1.0, "R"), (-1.0, "T")):
        cosT = (sin[:, None] * np.cos(phi)[None, :] * din[0] + sin[:, None] * np.sin(phi)[None, :] * din[1]
                + (sign * mu)[:, None] * din[2])
        pm = phase(cosT).mean(axis=1) / 2.0              # int dphi p / (4 pi) per unit mu
        depth = tt if sign > 0 else tau - tt
        esc = np.exp(-depth[:, None] / mu[None, :])
        inner = (esc * pm[None, :]).mean(axis=1)         # int_0^1 dmu
        out[name] = float((np.exp(-tt / mu0) / mu0 * inner).mean() * tau)
    return out["R"], out["T"]


@pytest.mark.parametrize("kind", ["rayleigh", "hg"])
def test_single_scatter_thin_slab(kind):
    """Photons whose record shows exactly ONE real scatter and no surface hit, leaving through the top
    (or absorbed at the black surface), against the first-order quadrature.  Slant sun, so the rotated
    direction's vertical component (the -s r cos(phi) + c mu formula) is what is being checked."""
    # Rayleigh: near 55 deg the hemispheric integrals of 3/4 (1 + cos^2) and of an isotropic phase function
    # coincide; at 15 deg they differ by 1.5 %, which 2^23 photons resolve (4 sigma = 0.9 %).
    tau, azi, g = 0.05, 140.0, 0.85
    zen = 55.0 if kind == "hg" else 15.0
    nz, dz = 8, 100.0
    cfg, opt = plane_parallel(8, 8, nz, 100.0, 100.0, dz, tau / (nz * dz), 1.0, g=g,
                              cloud_frac=1.0 if kind == "hg" else 0.0, albedo=0.0)
    n = 1 << (21 if kind == "hg" else 23)
    t, rec, _ = O.trace(cfg.grid, opt, zen, azi, n, seed=21, records=True, n_threads=T)
    tau32 = float(opt["k_ext"][0, 0, 0]) * nz * dz
    if kind == "hg":
        g32 = float(np.float32(g))
        phase = lambda c: (1 - g32 ** 2) / (1 + g32 ** 2 - 2 * g32 * c) ** 1.5
        assert t.counters.n_rayleigh == 0 and t.counters.n_hg > 0
    else:
        phase = lambda c: 0.75 * (1 + c ** 2)
        assert t.counters.n_hg == 0 and t.counters.n_rayleigh > 0
    R1, T1 = _single_scatter_quadrature(phase, tau32, zen, azi)
    fate, n_sfc, n_sc = rec[:, 0] & 0xFF, rec[:, 0] >> 8, rec[:, 3]
    r_obs = float(((n_sc == 1) & (fate == O.FATE_TOD_EXIT) & (n_sfc == 0)).mean())
    t_obs = float(((n_sc == 1) & (fate == O.FATE_SFC_ABS)).mean())
    within(r_obs, R1, n, extra=1e-3 * R1)
    within(t_obs, T1, n, extra=1e-3 * T1)
    # zeroth order for completeness: unscattered transmission
    within(float(((n_sc == 0) & (fate == O.FATE_SFC_ABS)).mean()), np.exp(-tau32 / np.cos(np.radians(zen))), n)
    assert int(t.atm_abs.sum()) == 0


@pytest.mark.parametrize("azi,axis,sign", [(0.0, 0, -1), (90.0, 1, -1), (180.0, 0, +1), (270.0, 1, +1)])
def test_cloud_shadow_displacement(azi, axis, sign):
    """BASELINE.json configs[0]: the cube's direct-beam shadow is displaced by h tan(theta0) away from the
    sun ("shadows ... horizontally shifted"); azimuth is the sun's position clockwise from north
    (P:64), x = east, y = north: sun in the north (0 deg) -> shadow towards -y, sun in the east -> -x."""
    cfg = CONFIGS[1]
    opt = make_optics(cfg)
    n = cfg.ncol * 64
    t, _, _ = O.trace(cfg.grid, opt, 30.0, azi, n, seed=1, n_threads=T)
    d = t.sfc_dir.astype(np.float64)
    deficit = np.clip(d.max() - d, 0, None)
    deficit[deficit < 0.5 * deficit.max()] = 0
    ang = 2 * np.pi * (np.arange(32) + 0.5) / 32
    w = deficit.sum(axis=1 - axis) if axis == 0 else deficit.sum(axis=0)
    centroid = (np.angle((w * np.exp(1j * ang)).sum()) % (2 * np.pi)) / (2 * np.pi) * 32   # voxel units
    # cube centre column 16.0, centre height 800 m: displacement 800 tan(30 deg) / 50 m = 9.24 voxels
    expect = (16.0 + sign * 800.0 * np.tan(np.radians(30.0)) / 50.0) % 32
    assert abs((centroid - expect + 16) % 32 - 16) < 0.75, (centroid, expect)
    # and the other axis is not displaced
    w2 = deficit.sum(axis=axis) if axis == 0 else deficit.sum(axis=1)
    c2 = (np.angle((w2 * np.exp(1j * ang)).sum()) % (2 * np.pi)) / (2 * np.pi) * 32
    assert abs(c2 - 16.0) < 0.75, c2
