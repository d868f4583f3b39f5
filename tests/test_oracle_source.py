"""Pins for the oracle's top-of-domain source options (NEXT-2): "Rays are initialized at
the domain top following a scrambled Sobol sequence ... Depending on the diffuse fraction, the initial direction
of each photon is either along the sun beam or randomly generated, assuming isotropic downwelling diffuse
radiation at the TOD."  Pinned against the net property of the Sobol sequence, exact balance of dyadic
strata through the tracer, and closed forms for the diffuse source."""
import numpy as np
from scipy import special

import oracle as O
from rt_inputs import plane_parallel
from test_oracle_pins import T, W0, frac, within


def test_sobol_points_are_a_net():
    """The first 2^m points of the 2-D Sobol sequence form a (0, m, 2)-net: every elementary interval
    [a 2^-p, (a+1) 2^-p) x [b 2^-q, (b+1) 2^-q) with p + q = m holds exactly one point; and a digital shift
    (XOR with any constant) keeps the property."""
    for m in (4, 7, 10):
        n = 1 << m
        x1, x2 = O.sobol2(np.arange(n))
        assert len(set(zip(x1.tolist(), x2.tolist()))) == n
        for shift in ((0, 0), (0x9E3779B9, 0x7F4A7C15)):
            a1, a2 = x1 ^ np.uint32(shift[0]), x2 ^ np.uint32(shift[1])
            for p in range(m + 1):
                q = m - p
                cell = (a1.astype(np.uint64) >> np.uint64(32 - p) if p else np.zeros(n, np.uint64)) * np.uint64(1 << q) \
                    + (a2.astype(np.uint64) >> np.uint64(32 - q) if q else np.zeros(n, np.uint64))
                assert np.array_equal(np.sort(cell), np.arange(n, dtype=np.uint64)), (m, p, shift)
    # the first coordinate is the radical inverse: point 1 = 1/2, point 2 = 1/4, point 3 = 3/4
    x1, x2 = O.sobol2(np.array([0, 1, 2, 3]))
    assert x1.tolist() == [0, 1 << 31, 1 << 30, 3 << 30] and x2.tolist() == [0, 1 << 31, 3 << 30, 1 << 30]


def _vacuum(nx, ny, nz, dx, dz):
    return plane_parallel(nx, ny, nz, dx, dx, dz, 0.0, 0.0, albedo=0.0, block=(2, 2, 2))


def test_sobol_entry_points_balance_dyadic_strata_exactly():
    """Vacuum, sun in the west at tan(theta0) = 2.5 dx / H: a photon entering column c at sub-pixel u lands in
    column c + 2 if u < 1/2 and c + 3 otherwise.  With 2^10 Sobol passes per column each half holds exactly
    half of the points, so every column receives exactly 2^10 photons; with the Philox entry points the same
    count fluctuates binomially (sigma = 16).  Shows that pass k of a column uses point k and that the scramble
    is a digital shift."""
    nx, ny, nz, dx, dz = 8, 4, 4, 100.0, 100.0
    cfg, opt = _vacuum(nx, ny, nz, dx, dz)
    zen = float(np.degrees(np.arctan(2.5 * dx / (nz * dz))))
    passes = 1 << 10
    n = nx * ny * passes
    ts, _, _ = O.trace(cfg.grid, opt, zen, 270.0, n, seed=3, n_threads=T, sobol=True)
    tp, _, _ = O.trace(cfg.grid, opt, zen, 270.0, n, seed=3, n_threads=T)
    cs = ts.sfc_dir.astype(np.int64) // W0
    cp = tp.sfc_dir.astype(np.int64) // W0
    assert cs.sum() == n and cp.sum() == n
    assert np.abs(cs - passes).max() <= 2, cs          # 2: a point exactly on the stratum edge may round either way
    assert np.abs(cp - passes).max() > 16
    # another call (other first id) is scrambled independently but balanced just the same
    t2, _, _ = O.trace(cfg.grid, opt, zen, 270.0, n, first_photon_id=n, seed=3, n_threads=T, sobol=True)
    assert np.abs(t2.sfc_dir.astype(np.int64) // W0 - passes).max() <= 2


def test_diffuse_source_fraction_and_angular_law():
    """Vacuum: the diffuse share of the surface arrivals is the diffuse fraction (binomial), direct + diffuse =
    all.  Pure absorber of vertical optical depth tau: diffuse photons arrive with probability
    int 2 mu exp(-tau/mu) dmu = 2 E3(tau) (isotropic downwelling radiance), beam photons with exp(-tau/mu0)."""
    n = 1 << 19
    f = 0.3
    cfg, opt = _vacuum(8, 8, 8, 100.0, 100.0)
    t, _, _ = O.trace(cfg.grid, opt, 40.0, 20.0, n, seed=6, n_threads=T, diffuse_fraction=f)
    assert int(t.sfc_dir.sum()) + int(t.sfc_dif.sum()) == n * W0 and t.closure() == n * W0
    within(frac(t.sfc_dif, n), float(np.float32(f)), n)
    tau, zen, nz, dz = 0.5, 40.0, 8, 250.0
    cfg, opt = plane_parallel(8, 8, nz, 100.0, 100.0, dz, tau / (nz * dz), 0.0, albedo=0.0)
    t, _, _ = O.trace(cfg.grid, opt, zen, 20.0, n, seed=7, n_threads=T, diffuse_fraction=f)
    tau32 = float(opt["k_ext"][0, 0, 0]) * nz * dz
    f32 = float(np.float32(f))
    within(frac(t.sfc_dif, n), f32 * 2.0 * special.expn(3, tau32), n)
    within(frac(t.sfc_dir, n), (1 - f32) * np.exp(-tau32 / np.cos(np.radians(zen))), n)
    assert abs(2.0 * special.expn(3, tau32) - special.expn(2, tau32)) > 0.1     # uniform-in-mu would give E2
    # limits: fraction 0 is the default stream bit for bit; fraction 1 leaves no direct light
    a, ra, _ = O.trace(cfg.grid, opt, zen, 20.0, 1 << 14, seed=7, records=True)
    b, rb, _ = O.trace(cfg.grid, opt, zen, 20.0, 1 << 14, seed=7, records=True, diffuse_fraction=0.0, sobol=False)
    assert np.array_equal(ra, rb) and np.array_equal(a.atm_abs, b.atm_abs)
    c, _, _ = O.trace(cfg.grid, opt, zen, 20.0, 1 << 14, seed=7, diffuse_fraction=1.0)
    assert int(c.sfc_dir.sum()) == 0 and int(c.sfc_dif.sum()) > 0
