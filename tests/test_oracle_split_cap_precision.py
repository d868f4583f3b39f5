"""Pins for three parts of the oracle that had none: the paper's cloud-vs-gas scattering
probability, the event cap, and the attribution of fp32-vs-fp64 path differences to
floating-point rounding (BASELINE.json north_star: ">= 99.9 % of individual photon paths identical, with
divergences attributed to float rounding").  Nothing here compares the oracle with the CUDA path."""
import numpy as np
import pytest
from scipy import stats

import oracle as O
from rt_inputs import CONFIGS, make_optics, plane_parallel

W0 = O.W0
T = 8


# ------------------------------------------------------------------------------------------------
# P:56 "the relative probability of being scattered by a cloud droplet as opposed to a gas molecule is
# given by k_ext,cloud / k_ext"; DESIGN.md §3.4 (c1, c2, c3)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("f", [0.1, 0.3, 0.8])
@pytest.mark.parametrize("ssa", [1.0, 0.7])
def test_cloud_vs_gas_scattering_probability(f, ssa):
    """Homogeneous slab whose voxels all hold cloud and gas: of the scattering events a fraction
    fl32(k_cloud) / fl32(k_ext) must be Henyey-Greenstein (cloud) and the rest Rayleigh (gas), and of the real
    collisions a fraction 1 - omega0 must absorb, each within 4 binomial sigma.  A swapped branch
    (1 - f), the ratio of scattering coefficients, or a c2 built on the wrong base would fail it."""
    cfg, opt = plane_parallel(8, 8, 8, 50.0, 50.0, 50.0, k_ext=0.01, ssa=ssa, g=0.5, cloud_frac=f,
                              albedo=1.0 if ssa == 1.0 else 0.3, block=(4, 4, 4))
    n = 1 << 16
    t, _, _ = O.trace(cfg.grid, opt, 30.0, 40.0, n, seed=5, n_threads=T)
    c = t.counters
    n_sc = c.n_hg + c.n_rayleigh
    n_real = n_sc + c.n_atm_abs
    assert c.n_null == 0 and c.n_events == n_real       # homogeneous: the majorant is k_ext itself
    p = float(opt["k_ext_cloud"].flat[0]) / float(opt["k_ext"].flat[0])
    assert abs(p - f) < 1e-6
    assert abs(c.n_hg / n_sc - p) <= 4 * np.sqrt(p * (1 - p) / n_sc), (c.n_hg / n_sc, p)
    pa = 1.0 - float(opt["ssa"].flat[0])
    if pa == 0.0:
        assert c.n_atm_abs == 0
    else:
        assert abs(c.n_atm_abs / n_real - pa) <= 4 * np.sqrt(pa * (1 - pa) / n_real)
    assert t.closure() == n * W0


def test_cloud_vs_gas_split_in_weighted_mode():
    """The same ratio in the paper's weighted mode, where absorption is a deposit and the event type is
    drawn among the non-absorbing outcomes only: HG : Rayleigh must still be k_cloud : k_gas-part, i.e. the HG
    share of the scatterings is (c2 - c1) / (c3 - c1) = omega0 k f / (omega0 k) = f."""
    f, ssa = 0.3, 0.7
    cfg, opt = plane_parallel(8, 8, 8, 50.0, 50.0, 50.0, k_ext=0.01, ssa=ssa, g=0.5, cloud_frac=f, albedo=0.3,
                              block=(4, 4, 4))
    n = 1 << 15
    t, _, _ = O.trace(cfg.grid, opt, 30.0, 40.0, n, seed=6, n_threads=T, weighted=True)
    c = t.counters
    n_sc = c.n_hg + c.n_rayleigh
    assert abs(c.n_hg / n_sc - f) <= 4 * np.sqrt(f * (1 - f) / n_sc)
    assert t.closure() == n * W0


# ------------------------------------------------------------------------------------------------
# "e > 2^20: stop, n_capped += 1, capped_energy += W0"
# ------------------------------------------------------------------------------------------------
def _cap_field(k_hat):
    """One acceleration cell of 8^3 voxels over the whole domain; a single dense voxel (in a column the
    vertical beam of the launched photons never enters) sets the majorant, every other voxel is EMPTY, so a
    photon meets nothing but null collisions, Poisson with mean k_hat x 400 m on its way to the surface."""
    k = np.zeros((8, 8, 8), np.float32)
    k[3, 7, 7] = k_hat
    opt = {"k_ext": k, "k_ext_cloud": np.zeros_like(k), "ssa": np.ones_like(k), "g": np.zeros_like(k),
           "sfc_albedo": np.zeros((8, 8), np.float32)}
    return (8, 8, 8, 50.0, 50.0, 50.0, 8, 8, 8), opt


@pytest.mark.parametrize("weighted", [False, True])
@pytest.mark.parametrize("precision", [64, 32])
def test_event_cap_every_photon(weighted, precision):
    """k_hat x 400 m = 1.2e6 expected null collisions, 138 sigma above the cap of 2^20: every photon must stop
    at the cap with exactly 2^20 counted events (the capped event itself is counted), fate 4, and its energy must
    go to capped_energy so that closure stays exact."""
    grid, opt = _cap_field(3000.0)
    n = 48                                              # columns 0..47: rows 0..5, never the dense voxel's column
    t, rec, _ = O.trace(grid, opt, 0.0, 0.0, n, seed=3, precision=precision, records=True, n_threads=T, weighted=weighted)
    c = t.counters
    assert c.n_capped == n and c.capped_energy == n * W0
    assert (rec[:, 0] == O.FATE_CAPPED).all() and (rec[:, 2] == 1 << 20).all() and (rec[:, 3] == 0).all()
    assert c.n_events == n << 20 and c.n_null == n << 20
    assert c.n_sfc_hits == 0 and c.n_toa == 0 and c.n_atm_abs == 0
    assert int(t.atm_abs.sum()) == 0 and int(t.sfc_abs.sum()) == 0 and t.closure() == n * W0


def test_event_cap_threshold_is_exact():
    """With k_hat x 400 m = 2^20 - 512 the number N of null collisions on the way down is Poisson(lambda) and a
    photon is capped iff N >= 2^20 (it stops when the event index would exceed 2^20): the capped share must be
    P(N >= 2^20) = 0.31 within 4 binomial sigma, every capped record must show exactly 2^20 events and every
    other photon fewer, ending in the (black) surface."""
    lam = float((1 << 20) - 512)
    k_hat = np.float32(lam / 400.0)
    lam = float(k_hat) * 400.0
    grid, opt = _cap_field(k_hat)
    n = 48 * 4
    t, rec, _ = O.trace(grid, opt, 0.0, 0.0, n, seed=11, records=True, n_threads=T)
    p = float(stats.poisson.sf((1 << 20) - 1, lam))
    capped = rec[:, 0] == O.FATE_CAPPED
    assert abs(capped.mean() - p) <= 4 * np.sqrt(p * (1 - p) / n), (capped.mean(), p)
    assert (rec[capped, 2] == 1 << 20).all()
    assert ((rec[~capped, 0] & 0xFF) == O.FATE_SFC_ABS).all() and (rec[~capped, 2] < 1 << 20).all()
    assert t.counters.n_capped == int(capped.sum()) and t.counters.capped_energy == int(capped.sum()) * W0
    assert t.closure() == n * W0


# ------------------------------------------------------------------------------------------------
# fp32 vs fp64: which photons differ, and why
# ------------------------------------------------------------------------------------------------
def first_differences(t_a, t_b):
    """From two decision logs: per photon the index of the first decision whose (kind, outcome) differs (-1 if the
    common part of the logs agrees), and whether the log was long enough to tell."""
    ca, ma, na = t_a.decisions
    cb, mb, nb = t_b.decisions
    K = ca.shape[1]
    L = np.minimum(np.minimum(na, nb), K)
    neq = (ca != cb) & (np.arange(K)[None, :] < L[:, None])
    has = neq.any(axis=1)
    first = np.where(has, neq.argmax(axis=1), -1)
    complete = (na <= K) & (nb <= K)
    return first, has, complete


@pytest.mark.parametrize("config,n_log2,min_same", [(1, 15, 0.9995), (2, 14, 0.994), (3, 13, 0.97)])
def test_fp32_vs_fp64_divergences_are_rounding(config, n_log2, min_same):
    """The kernel-precision instantiation (what the GPU must equal bit for bit) against the oracle proper on a
    sample of configs 1-3, with both runs logging every decision they take (kind, outcome, margin).
    Asserted: (1) the identical-path fraction (recorded in DESIGN.md §7); (2) a photon whose records differ shows a
    differing decision, and the fraction of photons with identical DECISION SEQUENCES (stricter than identical
    records: with voxel-sized cells a photon passing near a voxel edge may cross the two faces in the other order
    and still follow the same path) is within 3 % of it; (3) a photon whose records differ took the same decisions up to a first one, and
    at that one both runs faced the SAME kind of decision -- no difference in logic, only in which side of a
    threshold a rounded number fell; (4) the two runs' margins at agreeing decisions differ by rounding-scale
    amounts for the bulk of the decisions (median below 1e-5 of a voxel / cell), so the flipped decisions are the
    tail of a continuous rounding drift (amplified where DESIGN.md §7 says: optical depth carried from a cloud into
    clear air, grazing directions), not a second population."""
    cfg = CONFIGS[config]
    opt = make_optics(cfg)
    n = 1 << n_log2
    K = 8192
    kw = dict(seed=cfg.seed, records=True, n_threads=T, decision_log=K, **cfg.accel)
    t64, r64, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, precision=64, **kw)
    t32, r32, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, precision=32, **kw)
    same = (r64 == r32).all(axis=1)
    print("config %d: identical fp32/fp64 paths %.5f of %d" % (config, same.mean(), n))
    assert same.mean() >= min_same
    first, has, complete = first_differences(t64, t32)
    assert complete.mean() > 0.98                       # the log held nearly every photon's whole path
    # (2) the record criterion against the stricter one: every logged decision equal
    print("  identical decision sequences %.5f (records are a summary: a path may differ in between and still "
          "end in the same bin with the same counts)" % (~has)[complete].mean())
    assert (same | has)[complete].all() and (~has)[complete].mean() >= min_same - 0.03
    # (3) different records => a first differing decision, of the same kind in both runs
    d = np.where(~same & complete)[0]
    assert has[d].all()
    c64, m64, _ = t64.decisions
    c32, m32, _ = t32.decisions
    k = first[d]
    assert ((c64[d, k] >> 4) == (c32[d, k] >> 4)).all()
    # (4) rounding-scale drift where the decisions agree: margins of the floor-type decisions (in voxels)
    agree = (c64 == c32) & (np.arange(K)[None, :] < np.where(has, first, np.minimum(t64.decisions[2], K))[:, None])
    floors = agree & ((c64 >> 4) == O.DK_VOXEL)
    drift = np.abs(m64[floors].astype(np.float64) - m32[floors].astype(np.float64))
    assert drift.size > 1000
    print("  |margin64 - margin32| at agreeing voxel decisions: median %.2e, 90 %% %.2e, 99 %% %.2e" %
          (np.median(drift), np.percentile(drift, 90), np.percentile(drift, 99)))
    # the bulk is at rounding scale; the tail is the amplification DESIGN.md §7 derives: a path-length difference of
    # 1 mm inside a cloud (k = 0.1 / m) is 1e-4 of optical depth, i.e. 4 m of flight in the clear air below it
    # (k = 2.7e-5 / m), so voxel decisions in clear air see the largest drifts
    assert np.median(drift) < 1e-5 and np.percentile(drift, 99) < 0.5
