"""Acceptance of the CUDA path against the ORACLE PROPER (fp64) on all five configs (BASELINE.json north_star:
"energy closure bit-exact in fixed point and domain-mean fluxes within 4 Monte Carlo sigma ... per-voxel heating and
per-column irradiance RMS relative differences below 2 % where the tally holds >= 10^4 photon hits"; surface
fluxes and 3-D heating are what the tracer produces), plus the paths round 1 left without a GPU test: the event cap,
the generic pack kernel, the state errors of the slot API, job-indexed shards.  Everything goes through the C ABI."""
import numpy as np
import pytest
import torch

import oracle as O
from rt_inputs import CONFIGS, make_optics, plane_parallel, spectral_points

pytestmark = pytest.mark.gpu
NAMES = ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up")
T = 16


def _rt():
    import paper_2208_05247_b200 as rt
    return rt


def block_sums(a, blk):
    a = np.asarray(a, dtype=np.float64) / O.W0
    for ax, s in enumerate(blk):
        shp = list(a.shape)
        shp[ax:ax + 1] = [shp[ax] // s, s]
        a = a.reshape(shp).sum(axis=ax + 1)
    return a


def block_rms(gpu, ref, blk, min_hits=10_000):
    """RMS relative difference over the block sums of `ref` holding >= min_hits photon hits; and how many there are."""
    a, b = block_sums(gpu, blk), block_sums(ref, blk)
    m = b >= min_hits
    return (float(np.sqrt(np.mean(((a[m] - b[m]) / b[m]) ** 2))) if m.any() else None), int(m.sum())


def finest_block(ref, min_hits, min_blocks):
    """The finest (z, y, x) block, halving from the whole domain, that still leaves >= min_blocks blocks of `ref` with
    >= min_hits hits: the resolution at which the north_star's ">= 10^4 photon hits" criterion can be evaluated."""
    blk = list(ref.shape)
    best = None
    while True:
        b = block_sums(ref, blk)
        if int((b >= min_hits).sum()) >= min_blocks:
            best = tuple(blk)
        elif best is not None:
            return best
        ax = int(np.argmax(blk))                       # halve the longest extent
        if blk[ax] == 1 or (best is None and max(blk) <= 2):
            return best
        blk[ax] //= 2


def accept(cfg, opt, n, heat_blk=None, col_blk=(8, 8), stream_id=0, min_blocks=4, heat_min_hits=10_000, weighted=False):
    """GPU and fp64 oracle on the same n photon ids: closure, 4-sigma domain means, < 2 % block RMS of the surface
    irradiance AND the heating over blocks with >= 1e4 hits (the block sizes are chosen so that such blocks exist:
    a test over no block would be vacuous; heat_blk = None takes the finest block size that leaves min_blocks of
    them); returns the identical-record fraction."""
    rt = _rt()
    g = rt.Grid(*cfg.grid, device=0, **cfg.accel)
    g.set_mode(weighted)
    g.set_optics(opt["k_ext"], opt["k_ext_cloud"], opt["ssa"], opt["g"], opt["sfc_albedo"])
    rec = g.trace(cfg.zenith_deg, cfg.azimuth_deg, n, seed=cfg.seed, stream_id=stream_id, records=True)
    t = g.read_tallies()
    rec = rec.cpu().numpy().view(np.uint32)
    g.close()
    o64, rec64, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=cfg.seed, stream_id=stream_id,
                            precision=64, records=True, n_threads=T, weighted=weighted, **cfg.accel)
    assert t.closure() == n * rt.W0 and o64.closure() == n * rt.W0      # the roulette ledger included (weighted)
    assert t.counters.n_capped == 0 and t.counters.n_photons == n
    for name in NAMES:
        pg = float(getattr(t, name).sum()) / (n * rt.W0)
        po = float(getattr(o64, name).sum()) / (n * rt.W0)
        sigma = np.sqrt(max(po * (1 - po), 1e-12) / n)     # binomial: an upper bound for the weighted estimator too
        assert abs(pg - po) <= 4 * sigma, (name, pg, po, sigma)
    sfc_g = t.sfc_dir.numpy() + t.sfc_dif.numpy()
    sfc_o = o64.sfc_dir + o64.sfc_dif
    if col_blk is None:
        col_blk = finest_block(sfc_o, 10_000, min_blocks)
        assert col_blk is not None, "no block of columns with 1e4 surface hits at any resolution"
    rms_s, nb_s = block_rms(sfc_g, sfc_o, col_blk)
    if heat_blk is None:
        heat_blk = finest_block(o64.atm_abs, heat_min_hits, min_blocks)
        assert heat_blk is not None, "no heating block with %d hits at any resolution" % heat_min_hits
    rms_h, nb_h = block_rms(t.atm_abs.numpy(), o64.atm_abs, heat_blk, heat_min_hits)
    same = float((rec == rec64).all(axis=1).mean())
    assert nb_s >= min_blocks and nb_h >= min_blocks, (nb_s, nb_h)      # not vacuous
    print("%s: identical fp64 records %.5f; surface irradiance %d blocks of %s rms %.4f %%; heating %d blocks of %s rms %.4f %%"
          % (cfg.name, same, nb_s, col_blk, 100 * rms_s, nb_h, heat_blk, 100 * rms_h))
    assert rms_s < 0.02 and rms_h < 0.02, (rms_s, rms_h)
    return same


def test_acceptance_config1_full():
    """Config 1 absorbs ~9000 of its 2^18 photons in the whole atmosphere, so no heating bin of any size holds 1e4
    hits: the heating is compared per 8-level slab holding >= 1000 hits (RMS bar unchanged)."""
    cfg = CONFIGS[1]
    same = accept(cfg, make_optics(cfg), cfg.n_photons, heat_blk=(8, 32, 32), heat_min_hits=1000)
    assert same >= 0.999                                    # north_star's path-identity bar, against fp64


def test_acceptance_config2_full():
    cfg = CONFIGS[2]
    same = accept(cfg, make_optics(cfg), cfg.n_photons)
    assert same >= 0.995                                    # what fp32 geometry reaches on this field


def test_acceptance_config3_quarter():
    """2^24 photons (64 per column) of the bench workload in the bench's launch configuration."""
    cfg = CONFIGS[3]
    same = accept(cfg, make_optics(cfg), 1 << 24, col_blk=(16, 16))
    assert same >= 0.97                                     # DESIGN.md §7 (voxel-sized cells: more face decisions per photon)


def test_acceptance_config4_three_points():
    """Three spectral points of the sweep (clear-sky absorbing, mid, strongly absorbing cloud), each on its own
    stream id, 2^22 photons."""
    from dataclasses import replace
    cfg = CONFIGS[4]
    pts = spectral_points(112)
    for j in (3, 56, 108):
        opt = make_optics(cfg, pts[j])
        accept(replace(cfg, name="%s point %d" % (cfg.name, j)), opt, 1 << 22, col_blk=None, stream_id=j)


def test_acceptance_weighted_mode_configs_2_and_3():
    """The paper's own scheme (weights + Russian roulette) against the fp64 oracle in the
    same mode: config 2 in full and 2^22 photons of config 3 (closure with the roulette ledger, domain means, block
    RMS of irradiance and heating; "hits" are deposited quanta / W0)."""
    cfg = CONFIGS[2]
    accept(cfg, make_optics(cfg), cfg.n_photons, weighted=True)
    cfg = CONFIGS[3]
    accept(cfg, make_optics(cfg), 1 << 22, col_blk=(32, 32), weighted=True)


def test_acceptance_config5_sample():
    """1024x1024x192: 2^24 photons (16 per column)."""
    cfg = CONFIGS[5]
    same = accept(cfg, make_optics(cfg), 1 << 24, col_blk=(32, 32))
    assert same >= 0.96


# ------------------------------------------------------------------------------------------------------------
def _cap_field(k_hat):
    k = np.zeros((8, 8, 8), np.float32)
    k[3, 7, 7] = k_hat
    opt = {"k_ext": k, "k_ext_cloud": np.zeros_like(k), "ssa": np.ones_like(k), "g": np.zeros_like(k),
           "sfc_albedo": np.zeros((8, 8), np.float32)}
    return (8, 8, 8, 50.0, 50.0, 50.0, 8, 8, 8), opt


@pytest.mark.parametrize("weighted", [False, True])
def test_event_cap_on_gpu(weighted):
    """DESIGN.md §3.12 on the GPU (tests/test_oracle_split_cap_precision.py pins the oracle side): with
    k_hat x 400 m = 2^20 - 512 expected null collisions about a third of the photons reach the cap; fates,
    event counts, n_capped, capped_energy and closure must equal the oracle's in kernel precision."""
    rt = _rt()
    k_hat = np.float32(((1 << 20) - 512) / 400.0)
    grid, opt = _cap_field(k_hat)
    n = 48 * 4
    g = rt.Grid(*grid, device=0)
    g.set_mode(weighted)
    g.set_optics(opt["k_ext"], opt["k_ext_cloud"], opt["ssa"], opt["g"], opt["sfc_albedo"])
    rec = g.trace(0.0, 0.0, n, seed=11, records=True).cpu().numpy().view(np.uint32)
    t = g.read_tallies()
    g.close()
    o, rec32, _ = O.trace(grid, opt, 0.0, 0.0, n, seed=11, precision=32, records=True, n_threads=T, weighted=weighted)
    assert np.array_equal(rec, rec32)
    assert t.counters.asdict() == o.counters.asdict()
    capped = rec[:, 0] == rt.FATE_CAPPED
    assert 0 < capped.sum() < n and (rec[capped, 2] == 1 << 20).all()
    assert t.counters.n_capped == int(capped.sum()) and t.counters.capped_energy == int(capped.sum()) * rt.W0
    assert t.closure() == n * rt.W0


def test_generic_pack_kernel_odd_row_length_and_unaligned_views():
    """nx = 30 (not a multiple of 4) and field views that start 4 bytes into their allocation: rt_set_optics takes the
    one-thread-per-voxel pack kernel; packed records, majorant table (merged cells on) and a traced sample must
    equal the oracle's."""
    rt = _rt()
    nx, ny, nz = 30, 20, 16
    rng = np.random.default_rng(5)
    k = (1e-4 + 2e-2 * (rng.uniform(size=(nz, ny, nx)) < 0.15) * rng.uniform(0.2, 1.0, size=(nz, ny, nx))).astype(np.float32)
    kc = np.where(k > 1e-3, k - np.float32(1e-4), 0).astype(np.float32)
    opt = {"k_ext": k, "k_ext_cloud": kc, "ssa": np.where(k > 1e-3, 0.98, 0.5).astype(np.float32),
           "g": np.full(k.shape, 0.8, np.float32), "sfc_albedo": rng.uniform(0, 0.6, size=(ny, nx)).astype(np.float32)}
    grid = (nx, ny, nz, 40.0, 50.0, 30.0, 3, 2, 2)
    accel = {"merge": (2, 2, 2), "merge_ratio": 1.25}
    dev = torch.device("cuda", 0)
    views = {}
    for name, a in opt.items():
        buf = torch.zeros(a.size + 1, dtype=torch.float32, device=dev)
        buf[1:] = torch.from_numpy(a.ravel()).to(dev)
        views[name] = buf[1:]                                   # 4-byte offset: not 16-byte aligned
        assert views[name].data_ptr() % 16 == 4
    g = rt.Grid(*grid, device=0, **accel)
    g.set_optics(views["k_ext"], views["k_ext_cloud"], views["ssa"], views["g"], views["sfc_albedo"])
    packed = g.read_packed_optics().numpy().reshape(-1, 4)
    assert np.array_equal(packed, O.pack_optics_f32(opt["k_ext"], opt["k_ext_cloud"], opt["ssa"], opt["g"]))
    assert np.array_equal(g.read_majorant().numpy().view(np.uint32),
                          O.majorant(nx, ny, nz, 3, 2, 2, opt["k_ext"], **accel).view(np.uint32))
    n = 20000
    rec = g.trace(40.0, 250.0, n, seed=2, records=True).cpu().numpy().view(np.uint32)
    t = g.read_tallies()
    g.close()
    o, rec32, _ = O.trace(grid, opt, 40.0, 250.0, n, seed=2, precision=32, records=True, n_threads=T, **accel)
    assert np.array_equal(rec, rec32) and t.counters.asdict() == o.counters.asdict()
    for name in NAMES:
        assert np.array_equal(getattr(t, name).numpy(), getattr(o, name)), name


def test_slot_state_and_per_slot_errors():
    """rt_set_merge invalidates every slot; rt_set_point(0) invalidates rt_trace's optics; a slot's
    range error is reported by the launch that reads it, names the slot, does not taint other slots, and is
    healed by setting the slot again; the slot calls need rt_set_slots."""
    rt = _rt()
    cfg = CONFIGS[1]
    opt = make_optics(cfg)
    dev = torch.device("cuda", 0)
    f = {k: torch.from_numpy(v).to(dev) for k, v in opt.items()}
    args = (f["k_ext"], f["k_ext_cloud"], f["ssa"], f["g"], f["sfc_albedo"])
    g = rt.Grid(*cfg.grid, device=0, merge=(2, 2, 2))
    with pytest.raises(rt.RtError, match="rt_set_slots"):
        g.trace_batch(30.0, 0.0, [100])
    with pytest.raises(rt.RtError, match="rt_set_slots"):
        g.set_optics_factored(0, f["k_ext_cloud"], np.zeros(cfg.nz, np.float32), np.zeros(cfg.nz, np.float32), 0.9, 0.8,
                              f["sfc_albedo"])
    g.set_slots(3)
    for j in range(3):
        g.set_optics_slot(j, *args)
    g.trace_batch(30.0, 0.0, [100, 100, 100])
    # (1) new merge factors: the slots' majorant tables are stale
    g.set_merge(4, 4, 2)
    with pytest.raises(rt.RtError, match="no optics"):
        g.trace_batch(30.0, 0.0, [100, 100, 100])
    for j in range(3):
        g.set_optics_slot(j, *args)
    g.trace_batch(30.0, 0.0, [100, 100, 100])
    # (2) a bad slot: reported when launched, by number; the other slots still trace; re-setting heals it
    bad_k = f["k_ext"].clone()
    bad_k[3, 3, 3] = float("nan")
    g.set_optics_slot(1, bad_k, f["k_ext_cloud"], f["ssa"], f["g"], f["sfc_albedo"])
    with pytest.raises(rt.RtError, match="slot 1"):
        g.trace_batch(30.0, 0.0, [100, 100, 100])
    g.trace_batch(30.0, 0.0, [100], first_point=0)
    g.trace_batch(30.0, 0.0, [100], first_point=2)
    g.set_optics(*args)                                     # slot 0, synchronous: must not clear slot 1's mask
    with pytest.raises(rt.RtError, match="slot 1"):
        g.trace_batch(30.0, 0.0, [100, 100], first_point=1)
    g.set_optics_slot(1, *args)
    g.reset_tallies()
    g.trace_batch(30.0, 0.0, [100, 100, 100])
    assert g.read_tallies().counters.n_photons == 300
    # (3) rt_set_point on slot 0 replaces slot 0's majorant: rt_trace must refuse until rt_set_optics
    g.trace(30.0, 0.0, 100)
    g.set_cloud(f["k_ext_cloud"])
    g.set_point(0, np.full(cfg.nz, 2e-5, np.float32), np.full(cfg.nz, 1e-5, np.float32), 0.999, 0.85, f["sfc_albedo"])
    with pytest.raises(rt.RtError, match="rt_set_optics"):
        g.trace(30.0, 0.0, 100)
    g.set_optics(*args)
    g.trace(30.0, 0.0, 100)
    g.close()


def test_job_indexed_shards_equal_the_single_call():
    """include/rt.h rt_trace_range (the multi-GPU shard call): three ragged ranges of one job, on three contexts as
    three GPUs would hold them, sum to the single rt_trace call bit for bit, records included (Sobol entry points
    and a remainder pass in play, ids beyond 2^32)."""
    rt = _rt()
    cfg = CONFIGS[2]
    opt = make_optics(cfg)
    n = 5 * cfg.ncol + 4321
    first = (1 << 34) + 17
    args = (opt["k_ext"], opt["k_ext_cloud"], opt["ssa"], opt["g"], opt["sfc_albedo"])
    one = rt.Grid(*cfg.grid, device=0, **cfg.accel)
    one.set_source(0.0, sobol=True)
    one.set_optics(*args)
    rec1 = one.trace(cfg.zenith_deg, cfg.azimuth_deg, n, first_photon_id=first, seed=7, records=True).cpu()
    t1 = one.read_tallies()
    one.close()
    cuts = [0, 3 * cfg.ncol + 11, 4 * cfg.ncol + 5, n]
    total = {k: 0 for k in NAMES}
    recs, counters = [], None
    for b, e in zip(cuts[:-1], cuts[1:]):
        g = rt.Grid(*cfg.grid, device=0, **cfg.accel)
        g.set_source(0.0, sobol=True)
        g.set_optics(*args)
        recs.append(g.trace_range(cfg.zenith_deg, cfg.azimuth_deg, n, b, e - b, first_photon_id=first, seed=7, records=True).cpu())
        t = g.read_tallies()
        for k in NAMES:
            total[k] = total[k] + getattr(t, k)
        c = t.counters.asdict()
        counters = c if counters is None else {k: counters[k] + v for k, v in c.items()}
        g.close()
    assert torch.equal(torch.cat(recs), rec1)
    for k in NAMES:
        assert torch.equal(total[k], getattr(t1, k)), k
    assert counters == t1.counters.asdict()
    with pytest.raises(rt.RtError):
        g2 = rt.Grid(*cfg.grid, device=0)
        g2.set_optics(*args)
        g2.trace_range(cfg.zenith_deg, cfg.azimuth_deg, 100, 90, 20)
