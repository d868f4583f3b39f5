"""BASELINE.json configs[3] (spectral sweep, 112 points on the 512x512x128 field) and configs[4] (convergence
sweep on 1024x1024x192) on the GPU, through the C ABI, against the oracle.

Whole sweeps are checked by what holds at any size (closure bit-exact in fixed point, counter identities,
no capped photon, the paper's N^-1/2 noise law); sampled launches are compared with the oracle in
kernel precision record by record and tally by tally."""
import numpy as np
import pytest
import torch

import oracle as O
from rt_inputs import CONFIGS, make_optics, make_optics_torch, spectral_points, split_photons

pytestmark = pytest.mark.gpu

NAMES = ("k_ext", "k_ext_cloud", "ssa", "g", "sfc_albedo")
TALLIES = ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up")


def _rt():
    import paper_2208_05247_b200 as rt
    return rt


def test_config4_spectral_sweep():
    rt = _rt()
    from paper_2208_05247_b200.sweeps import spectral_sweep
    cfg = CONFIGS[4]
    pts = spectral_points(112)
    counts = split_photons(cfg.n_photons, [p["weight"] for p in pts])
    assert sum(counts) == cfg.n_photons and len(counts) == 112 and min(counts) > 0
    g = rt.Grid(*cfg.grid, device=0, **cfg.accel)

    # the device-side field assembly hands the library the same fp32 arrays as the host recipe
    sample = (0, 37, 111)
    host_opt = {}
    for j in sample:
        host_opt[j] = make_optics(cfg, pts[j])
        dev = make_optics_torch(cfg, pts[j])
        for k in NAMES:
            assert np.array_equal(dev[k].cpu().numpy().view(np.uint32), host_opt[j][k].view(np.uint32)), (j, k)

    # sampled points: 2^17 photons each (not a multiple of ncol: all launch from random columns),
    # stream_id = j, against the oracle in kernel precision
    n = 1 << 17
    for j in sample:
        opt = host_opt[j]
        g.reset_tallies()
        g.set_optics(*[opt[k] for k in NAMES])
        rec = g.trace(cfg.zenith_deg, cfg.azimuth_deg, n, seed=cfg.seed, stream_id=j, records=True)
        t = g.read_tallies()
        o32, rec32, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=cfg.seed, stream_id=j,
                                precision=32, records=True, n_threads=8, **cfg.accel)
        assert np.array_equal(rec.cpu().numpy().view(np.uint32), rec32), j
        for name in TALLIES:
            assert np.array_equal(getattr(t, name).numpy(), getattr(o32, name)), (j, name)
        assert t.counters.asdict() == o32.counters.asdict()
    del host_opt

    # the whole sweep: 112 x (rt_set_optics + rt_trace), tallies accumulated over the points
    g.reset_tallies()
    total = spectral_sweep(g, lambda j: [make_optics_torch(cfg, pts[j])[k] for k in NAMES], counts,
                           cfg.zenith_deg, cfg.azimuth_deg, seed=cfg.seed)
    t = g.read_tallies()
    c = t.counters
    assert total == cfg.n_photons and c.n_photons == total and c.n_capped == 0
    assert t.closure() == total * rt.W0
    assert c.n_events == c.n_null + c.n_rayleigh + c.n_hg + c.n_atm_abs
    assert int(t.sfc_dir.sum() + t.sfc_dif.sum()) == c.n_sfc_hits * rt.W0
    assert int(t.atm_abs.sum()) == c.n_atm_abs * rt.W0 and int(t.toa_up.sum()) == c.n_toa * rt.W0
    # a sweep in which many points absorb strongly: broadband absorption well above the single-point config 3
    assert 0.05 < c.n_atm_abs / total < 0.9

    # the same sweep over two contexts on two streams (points alternate, launches overlap): the summed integer
    # tallies and counters must equal the one-context sweep's exactly
    from paper_2208_05247_b200.sweeps import spectral_sweep_overlapped, sum_tallies
    g2 = rt.Grid(*cfg.grid, device=0, **cfg.accel)
    g.reset_tallies()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    total2 = spectral_sweep_overlapped([g, g2], streams, lambda j: [make_optics_torch(cfg, pts[j])[k] for k in NAMES],
                                       counts, cfg.zenith_deg, cfg.azimuth_deg, seed=cfg.seed)
    torch.cuda.synchronize()
    t2 = sum_tallies([g, g2], host=True)
    assert total2 == total and t2.counters.asdict() == c.asdict()
    for name in TALLIES:
        assert torch.equal(getattr(t2, name), getattr(t, name)), name
    g2.close()

    # ... and with all 112 points' optics resident in HBM slots and ONE launch (rt_trace_batch)
    from paper_2208_05247_b200.sweeps import spectral_sweep_batched
    g.set_slots(112)
    g.reset_tallies()
    total3 = spectral_sweep_batched(g, lambda j: [make_optics_torch(cfg, pts[j])[k] for k in NAMES], counts,
                                    cfg.zenith_deg, cfg.azimuth_deg, seed=cfg.seed)
    t3 = g.read_tallies()
    assert total3 == total and t3.counters.asdict() == c.asdict()
    for name in TALLIES:
        assert torch.equal(getattr(t3, name), getattr(t, name)), name
    # ... and as two launches over the two halves of the points (first_point), one after the other
    g.reset_tallies()
    g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts[:50], seed=cfg.seed)
    g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts[50:], seed=cfg.seed, first_point=50)
    t4 = g.read_tallies()
    assert t4.counters.asdict() == c.asdict()
    for name in TALLIES:
        assert torch.equal(getattr(t4, name), getattr(t, name)), name
    g.close()


def test_config5_convergence_sweep():
    rt = _rt()
    from paper_2208_05247_b200.sweeps import convergence_sweep
    cfg = CONFIGS[5]
    opt = make_optics(cfg)
    g = rt.Grid(*cfg.grid, device=0, **cfg.accel)
    g.set_optics(*[opt[k] for k in NAMES])

    # 1 photon per column (2^20 photons, one full pass) against the oracle in kernel precision
    n = cfg.ncol
    rec = g.trace(cfg.zenith_deg, cfg.azimuth_deg, n, seed=cfg.seed, records=True).cpu().numpy().view(np.uint32)
    t = g.read_tallies()
    o32, rec32, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=cfg.seed, precision=32,
                            records=True, n_threads=8, **cfg.accel)
    assert np.array_equal(rec, rec32)
    for name in TALLIES:
        assert np.array_equal(getattr(t, name).numpy(), getattr(o32, name)), name
    assert t.counters.asdict() == o32.counters.asdict()
    del t, o32, rec, rec32

    per_column = (1, 4, 16, 64, 256)
    rows, ref = convergence_sweep(g, cfg.ncol, per_column, cfg.zenith_deg, cfg.azimuth_deg, seed=cfg.seed,
                                  sfc_block=(16, 16), vox_block=(16, 32, 32), min_hits=500)
    print(rows)                                   # shown with pytest -s: the sweep table of DESIGN.md §6
    g.close()
    assert [r["photons_per_column"] for r in rows] == list(per_column)
    for r in rows:
        assert r["closure_exact"] and r["n_capped"] == 0
        assert r["sfc_blocks"] >= 1000 and r["heating_blocks"] >= 100
    # the noise falls as N^-1/2.  With an independent 256-per-column reference the expected RMS
    # difference is c sqrt(1/N + 1/256): c is the same at every N (15 % covers its own sampling error and
    # the non-Poisson part of the surface tally, whose direct beam is stratified by column)
    for key in ("rms_noise_sfc", "rms_noise_heating"):
        c = [r[key] / np.sqrt(1.0 / r["photons_per_column"] + 1.0 / ref["photons_per_column"]) for r in rows]
        assert max(c) / min(c) < 1.15, (key, c)
        assert rows[0][key] > 4 * rows[3][key]        # 64x the photons: ~ sqrt((1+1/256)/(1/64+1/256)) = 7.2
    # P:78 "the run time scales linearly with the number of samples": the same photons per second at 16, 64 and 256
    # photons per column (the 1- and 4-per-column launches last 2-8 ms, where the drain of the persistent kernel shows)
    pps = [r["paths_per_s"] for r in rows if r["photons_per_column"] >= 16]
    assert max(pps) / min(pps) < 1.15, pps
    assert rows[1]["paths_per_s"] > 0.6 * max(pps)


def test_batched_points_equal_separate_traces():
    """rt_trace_batch (one launch, slots in HBM) traces exactly what separate rt_trace calls per point would:
    records per point against the oracle in kernel precision (own optics, stream id = point, ragged counts incl.
    0 and a remainder pass), accumulated tallies and counters = the sum over the points."""
    rt = _rt()
    from dataclasses import replace
    cfg = replace(CONFIGS[2], block=(2, 2, 2), merge=(8, 8, 4))
    pts = spectral_points(112)
    sel = (3, 40, 77, 111, 5)
    counts = [cfg.ncol * 2 + 77, 0, 1000, cfg.ncol, 33]
    g = rt.Grid(*cfg.grid, device=0, **cfg.accel)
    g.set_slots(len(sel))
    opts = [make_optics(cfg, pts[j]) for j in sel]
    for k, opt in enumerate(opts):
        g.set_optics_slot(k, *[opt[n] for n in NAMES])
    first = (1 << 33) + 11
    for weighted in (False, True):
        g.reset_tallies()
        g.set_mode(weighted)
        rec = g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, first_photon_id=first, seed=cfg.seed,
                            records=True).cpu().numpy().view(np.uint32)
        t = g.read_tallies()
        total = O.Tallies(cfg.nx, cfg.ny, cfg.nz)
        off = 0
        for k, (opt, n) in enumerate(zip(opts, counts)):
            if n == 0:
                continue
            _, rec32, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, first_photon_id=first, seed=cfg.seed,
                                  stream_id=k, precision=32, records=True, n_threads=8, tallies=total,
                                  weighted=weighted, **cfg.accel)
            assert np.array_equal(rec[off:off + n], rec32), (k, weighted)
            off += n
        for name in TALLIES:
            assert np.array_equal(getattr(t, name).numpy(), getattr(total, name)), (name, weighted)
        assert t.counters.asdict() == total.counters.asdict() and t.closure() == sum(counts) * rt.W0
    # slot 0 is also what rt_set_optics / rt_trace use
    g.set_mode(False)
    g.reset_tallies()
    g.set_optics(*[opts[2][n] for n in NAMES])
    rec = g.trace(cfg.zenith_deg, cfg.azimuth_deg, 5000, seed=cfg.seed, stream_id=9, records=True).cpu().numpy().view(np.uint32)
    _, rec32, _ = O.trace(cfg.grid, opts[2], cfg.zenith_deg, cfg.azimuth_deg, 5000, seed=cfg.seed, stream_id=9,
                          precision=32, records=True, n_threads=8, **cfg.accel)
    assert np.array_equal(rec, rec32)
    # errors: a slot without optics, a bad field reported at the batch trace
    g.set_slots(2)
    g.set_optics_slot(0, *[opts[0][n] for n in NAMES])
    with pytest.raises(rt.RtError):
        g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, [10, 10])
    bad = opts[0]["ssa"].copy()
    bad[1, 2, 3] = -0.5
    g.set_optics_slot(1, opts[0]["k_ext"], opts[0]["k_ext_cloud"], bad, opts[0]["g"], opts[0]["sfc_albedo"])
    with pytest.raises(rt.RtError):
        g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, [10, 10])
    g.close()


def test_factored_optics_slots():
    """rt_set_optics_factored: packed optics and majorant table bit-identical to the oracle's
    packing of the fields assembled from the factors; a batched trace over factored slots identical to the oracle
    on those fields; bad factors are refused."""
    rt = _rt()
    from dataclasses import replace
    from rt_inputs import factored_point
    cfg = replace(CONFIGS[2], block=(2, 2, 2), merge=(8, 8, 4))
    pts = spectral_points(112)
    sel = (0, 58, 111)
    g = rt.Grid(*cfg.grid, device=0, **cfg.accel)
    g.set_slots(len(sel))
    facs = [factored_point(cfg, pts[j]) for j in sel]
    kc_dev = torch.from_numpy(facs[0]["k_cloud"]).cuda()
    al_dev = torch.from_numpy(facs[0]["sfc_albedo"]).cuda()
    fields = []
    for k, f in enumerate(facs):
        g.set_optics_factored(k, kc_dev, f["k_abs"], f["k_ray"], f["cloud_ssa"], f["cloud_g"], al_dev)
        asm = O.assemble_factored(f["k_cloud"], f["k_abs"], f["k_ray"], f["cloud_ssa"], f["cloud_g"])
        asm["sfc_albedo"] = f["sfc_albedo"]
        fields.append(asm)
    packed = g.read_packed_optics().numpy().reshape(-1, 4)           # slot 0
    want = O.pack_optics_f32(fields[0]["k_ext"], fields[0]["k_ext_cloud"], fields[0]["ssa"], fields[0]["g"])
    assert np.array_equal(packed.view(np.uint32), want.view(np.uint32))
    kh = g.read_majorant().numpy()
    assert np.array_equal(kh.view(np.uint32), O.majorant(cfg.nx, cfg.ny, cfg.nz, *cfg.block, fields[0]["k_ext"],
                                                         **cfg.accel).view(np.uint32))
    counts = [cfg.ncol + 99, 4000, cfg.ncol * 2]
    rec = g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, seed=cfg.seed, records=True).cpu().numpy().view(np.uint32)
    t = g.read_tallies()
    total = O.Tallies(cfg.nx, cfg.ny, cfg.nz)
    off = 0
    for k, (opt, n) in enumerate(zip(fields, counts)):
        _, rec32, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=cfg.seed, stream_id=k,
                              precision=32, records=True, n_threads=8, tallies=total, **cfg.accel)
        assert np.array_equal(rec[off:off + n], rec32), k
        off += n
    for name in TALLIES:
        assert np.array_equal(getattr(t, name).numpy(), getattr(total, name)), name
    assert t.counters.asdict() == total.counters.asdict()
    # the same points kept factored in the trace (rt_set_cloud + rt_set_point): no packed records at all; the
    # majorant table and every photon must come out the same
    g2 = rt.Grid(*cfg.grid, device=0, **cfg.accel)
    g2.set_slots(len(sel))
    with pytest.raises(rt.RtError):
        g2.set_point(0, facs[0]["k_abs"], facs[0]["k_ray"], facs[0]["cloud_ssa"], facs[0]["cloud_g"], al_dev)   # no cloud yet
    g2.set_cloud(facs[0]["k_cloud"])                                     # host field accepted
    for k, f in enumerate(facs):
        g2.set_point(k, f["k_abs"], f["k_ray"], f["cloud_ssa"], f["cloud_g"], f["sfc_albedo"])
    assert np.array_equal(g2.read_majorant().numpy().view(np.uint32), kh.view(np.uint32))
    # rt_set_points on cells of several voxels = the same calls point by point (slots 1, 2 set again that way)
    g2.set_points(1, np.stack([f["k_abs"] for f in facs[1:]]), np.stack([f["k_ray"] for f in facs[1:]]),
                  [f["cloud_ssa"] for f in facs[1:]], [f["cloud_g"] for f in facs[1:]], al_dev)
    for weighted in (False, True):
        g.reset_tallies(); g2.reset_tallies()
        g.set_mode(weighted); g2.set_mode(weighted)
        ra = g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, seed=cfg.seed, records=True)
        rb = g2.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, seed=cfg.seed, records=True)
        assert torch.equal(ra, rb), weighted
        ta, tb = g.read_tallies(), g2.read_tallies()
        for name in TALLIES:
            assert torch.equal(getattr(ta, name), getattr(tb, name)), (name, weighted)
        assert ta.counters.asdict() == tb.counters.asdict()
    g.set_mode(False)
    assert np.array_equal(rb.cpu().numpy().view(np.uint32)[:0], rec[:0])
    g2.close()
    with pytest.raises(rt.RtError):
        g.set_optics_factored(0, kc_dev, facs[0]["k_abs"], facs[0]["k_ray"], 1.5, 0.8, al_dev)
    with pytest.raises(rt.RtError):
        g.set_optics_factored(0, facs[0]["k_cloud"], facs[0]["k_abs"], facs[0]["k_ray"], 0.9, 0.8, al_dev)   # host field
    g.close()


@pytest.mark.parametrize("merge", [(8, 8, 8), (4, 2, 16)])
def test_points_on_voxel_sized_cells_keep_no_majorant_table(merge):
    """rt_set_cloud + rt_set_point on voxel-sized cells with merging: the library builds no majorant
    table per point; MOVE takes a voxel's majorant from the shared cloud field and the point's gas sums, and one word
    per block of merged cells says whether the block is merged.  Every photon must equal the oracle's on the fields
    assembled from the same factors (oracle: its own majorant table of voxel-sized cells), in both modes, with ragged
    counts; and a changed merge setting must ask for the cloud field again."""
    rt = _rt()
    from dataclasses import replace
    from rt_inputs import factored_point
    cfg = replace(CONFIGS[2], block=(1, 1, 1), merge=merge)
    pts = spectral_points(112)
    sel = (0, 58, 111, 30)
    facs = [factored_point(cfg, pts[j]) for j in sel]
    for k, f in enumerate(facs):                            # a different albedo per point
        f["sfc_albedo"] = np.clip(f["sfc_albedo"] * np.float32(0.5 + 0.25 * k), 0.0, 1.0).astype(np.float32)
    fields = []
    for f in facs:
        asm = O.assemble_factored(f["k_cloud"], f["k_abs"], f["k_ray"], f["cloud_ssa"], f["cloud_g"])
        asm["sfc_albedo"] = f["sfc_albedo"]
        fields.append(asm)
    g = rt.Grid(*cfg.grid, device=0, **cfg.accel)
    g.set_slots(len(sel))
    g.set_cloud(torch.from_numpy(facs[0]["k_cloud"]).cuda())
    for k, f in enumerate(facs):
        g.set_point(k, f["k_abs"], f["k_ray"], f["cloud_ssa"], f["cloud_g"], f["sfc_albedo"])
    with pytest.raises(rt.RtError):
        g.read_majorant()                                   # there is none in this mode
    counts = [cfg.ncol + 99, 4000, cfg.ncol * 2, 0]
    for weighted in (False, True):
        g.reset_tallies()
        g.set_mode(weighted)
        rec = g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, seed=cfg.seed, records=True).cpu().numpy().view(np.uint32)
        t = g.read_tallies()
        total = O.Tallies(cfg.nx, cfg.ny, cfg.nz)
        off = 0
        for k, (opt, n) in enumerate(zip(fields, counts)):
            if n == 0:
                continue
            _, rec32, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, seed=cfg.seed, stream_id=k,
                                  precision=32, records=True, n_threads=8, tallies=total, weighted=weighted, **cfg.accel)
            assert np.array_equal(rec[off:off + n], rec32), (k, weighted)
            off += n
        for name in TALLIES:
            assert np.array_equal(getattr(t, name).numpy(), getattr(total, name)), (name, weighted)
        assert t.counters.asdict() == total.counters.asdict() and t.closure() == sum(counts) * rt.W0
        assert t.counters.n_relevel > 0                     # both levels were in use
    # rt_set_points: the same slots in ONE call trace the same photons (weighted mode is still on), with one albedo
    # per point and with one albedo for all points
    g3 = rt.Grid(*cfg.grid, device=0, **cfg.accel)
    g3.set_slots(len(sel))
    g3.set_mode(True)
    g3.set_cloud(facs[0]["k_cloud"])
    ka, kr = np.stack([f["k_abs"] for f in facs]), np.stack([f["k_ray"] for f in facs])
    ssa, cg = [f["cloud_ssa"] for f in facs], [f["cloud_g"] for f in facs]
    g3.set_points(0, ka, kr, ssa, cg, torch.from_numpy(np.stack([f["sfc_albedo"] for f in facs])).cuda())
    rec3 = g3.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, seed=cfg.seed, records=True).cpu().numpy().view(np.uint32)
    assert np.array_equal(rec3, rec)
    t3 = g3.read_tallies()
    for name in TALLIES:
        assert torch.equal(getattr(t3, name), getattr(t, name)), name
    g3.reset_tallies(); g.reset_tallies()
    g3.set_points(1, ka[1:], kr[1:], ssa[1:], cg[1:], facs[2]["sfc_albedo"])          # host albedo, shared; slots 1..3
    for k in range(1, len(sel)):
        f = facs[k]
        g.set_point(k, f["k_abs"], f["k_ray"], f["cloud_ssa"], f["cloud_g"], facs[2]["sfc_albedo"])
    ra = g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, seed=cfg.seed, records=True)
    rb = g3.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, seed=cfg.seed, records=True)
    assert torch.equal(ra, rb) and not np.array_equal(rb.cpu().numpy().view(np.uint32), rec)
    with pytest.raises(rt.RtError):
        g3.set_points(2, ka, kr, ssa, cg, facs[0]["sfc_albedo"])                      # 4 points from slot 2 of 4
    with pytest.raises(rt.RtError):
        g3.set_points(0, ka, kr, [1.5] + ssa[1:], cg, facs[0]["sfc_albedo"])
    g3.close()
    # a bad cloud field is refused by rt_set_cloud in this mode too; new merge factors invalidate the cloud tables
    bad = facs[0]["k_cloud"].copy()
    bad[3, 4, 5] = -1.0
    with pytest.raises(rt.RtError):
        g.set_cloud(bad)
    g.set_cloud(facs[0]["k_cloud"])
    g.set_merge(2, 2, 2)
    with pytest.raises(rt.RtError):
        g.set_point(0, facs[0]["k_abs"], facs[0]["k_ray"], facs[0]["cloud_ssa"], facs[0]["cloud_g"], facs[0]["sfc_albedo"])
    g.close()
