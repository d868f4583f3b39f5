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


def test_rotation_geometry():
    """New direction d' is a unit vector with d . d' = mu; azimuth 2 pi u turns d' around d through a
    full circle (the perpendicular parts at u and u + 1/2 are opposite, at u + 1/4 orthogonal)."""
    rng = np.random.default_rng(11)
    for _ in range(300):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        if rng.uniform() < 0.15:
            d = np.array([1e-4 * rng.normal(), 1e-4 * rng.normal(), rng.choice([-1.0, 1.0])])
            d /= np.linalg.norm(d)          # the |c| >= 0.99999 branch
        mu, u = rng.uniform(-1, 1), rng.uniform(0, 0.5)
        a = O.rotate(d, mu, u)
        b = O.rotate(d, mu, u + 0.5)
        c = O.rotate(d, mu, u + 0.25)
        for v in (a, b, c):
            assert abs(np.linalg.norm(v) - 1) < 1e-12 and abs(v @ d - mu) < 1e-9
        pa, pb, pc = a - mu * d, b - mu * d, c - mu * d
        assert np.abs(pa + pb).max() < 1e-7 and abs(pa @ pc) < 1e-7


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
