"""bench.py — throughput of the photon-tracing hot path (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path over the 512x512x128 seeded
cumulus field (BASELINE.json configs[2]): rt_reset_tallies, rt_set_optics (pack + majorant),
rt_trace of 2^26 photons, rt_read_tallies (counters + the four column tallies; atm_abs stays on the
device for the device-timed value, and comes to the host in the e2e leg).  Prints ONE JSON line.

--impl reference times the CPU oracle (oracle/), as it stands, on a bounded sample of the same
workload on the box's host cores.  It is a deliberately slow checker, not a target.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

WORKLOAD = 3                      # default rt_inputs.CONFIGS key: BASELINE.json configs[2], 512x512x128 (the
                                  # configuration the metric is quoted on); --workload N times another config
METRIC = "photon_paths_per_s"
UNIT = "paths/s"
REF_SAMPLE_PHOTONS = 1 << 23      # per --impl reference step: 32 photons per column (~2 s on 16 cores)
CPU_BASELINE_PHOTONS = 1 << 25    # cpu_baseline leg: 128 photons per column (~10 s on 16 cores)
SECTOR = 32                       # bytes moved per random 16-byte gather (one DRAM/L2 sector)
COUNTERS_FILE = os.path.join(ROOT, "profiles", "trace_kernel_counters.json")   # ncu counters per workload (text)
KERNEL_SOURCES = ("rt_trace.cuh", "rt_device.cuh")   # what the trace kernel is compiled from: hashed into that file


def _kernel_sha16():
    """sha256 of the trace kernel's sources: an ncu entry only counts for the kernel it was captured from."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2208_05247_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def _ncu_counters(cfg, mode, n):
    """The committed ncu counters of the trace kernel for this workload, or None if there are none for the
    kernel as it stands (profiles/trace_kernel_counters.md says how they were captured)."""
    if not os.path.exists(COUNTERS_FILE):
        return None
    with open(COUNTERS_FILE) as f:
        entries = json.load(f).get("entries", [])
    sha = _kernel_sha16()
    for e in entries:
        if (e.get("workload") == cfg.name and e.get("mode") == mode and e.get("n_photons") == n
                and e.get("block") == list(cfg.block) and e.get("merge") == list(cfg.merge)
                and e.get("kernel_sha16") == sha):
            return e
    return None


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def _sm_max_mhz():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f).get("sm_max_mhz", 1965.0))
    return 1965.0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, uuid=None):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        cmd = ["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "200"]
        if uuid:
            cmd += ["-i", uuid]
        try:
            self.p = subprocess.Popen(cmd, stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for name, v in zip(names, parts[3:7]):
                if v.lower() == "active":
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def run_reference(args):
    """The oracle on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle as O
    from rt_inputs import CONFIGS, make_optics
    cfg = CONFIGS[args.workload if args.workload != 4 else 3]   # the spectral sweep's field is config 3's
    opt = make_optics(cfg)
    cores = O.hardware_threads()
    n = REF_SAMPLE_PHOTONS
    times, events = [], 0
    for step in range(args.warmup + args.steps):
        t, _, el = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, first_photon_id=step * n,
                           seed=cfg.seed, precision=64, n_threads=cores, weighted=(args.mode == "weighted"), **cfg.accel)
        assert t.closure() == n * O.W0
        if step >= args.warmup:
            times.append(el)
            events += t.counters.n_events
    total = sum(times)
    value = n * len(times) / total
    sample = "%d photons per step (%.0f per column) of the %d-photon workload, photon loop only" % (
        n, n / cfg.ncol, cfg.n_photons)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "collision_events_per_s": events / total,
        "config": {"workload": cfg.name, "grid": [cfg.nx, cfg.ny, cfg.nz], "photons_per_step": n,
                   "block": list(cfg.block), "zenith_deg": cfg.zenith_deg, "azimuth_deg": cfg.azimuth_deg},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2208_05247_b200 as rt          # raises if the CUDA library is missing: no CPU fallback
    from paper_2208_05247_b200.shard import weak_range
    from rt_inputs import CONFIGS, make_optics

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    cfg = CONFIGS[args.workload]
    if args.block:
        from dataclasses import replace
        cfg = replace(cfg, block=tuple(int(x) for x in args.block.split(",")))
    if args.merge:
        from dataclasses import replace
        cfg = replace(cfg, merge=tuple(int(x) for x in args.merge.split(",")))
    opt = make_optics(cfg)                       # seeded: every rank builds the same field
    names = ("k_ext", "k_ext_cloud", "ssa", "g", "sfc_albedo")
    spectral = args.workload == 4
    host = [torch.from_numpy(opt[k]).pin_memory() for k in names] if not spectral else None
    n = cfg.n_photons                            # per GPU (weak scaling: photon ids are sharded by rank)
    g = rt.Grid(*cfg.grid, device=local, **cfg.accel)
    g.set_mode(weighted=(args.mode == "weighted"))
    pinned_cols = rt.Tallies(None, *[torch.empty((cfg.ny, cfg.nx), dtype=torch.int64).pin_memory() for _ in range(4)],
                             counters=None)
    if spectral:
        # BASELINE.json configs[3]: 112 spectral points, each its own optics on the same cloud field, photons
        # split by irradiance weight; all 112 field sets resident in HBM (43 GB of the 180 GB) before timing
        from rt_inputs import make_optics_torch, spectral_points, split_photons
        from paper_2208_05247_b200.sweeps import spectral_sweep_overlapped
        pts = spectral_points(112)
        counts = split_photons(n, [p["weight"] for p in pts])
        factored = not args.full_fields and args.contexts == 0
        facs = None
        if factored:
            # FACTORED inputs (rt_set_optics_factored): one cloud field on the device + 2 nz numbers per point
            import numpy as np
            from rt_inputs import factored_point
            facs = [factored_point(cfg, p) for p in pts]
            kc_dev = torch.from_numpy(facs[0]["k_cloud"]).to(dev)
            al_dev = torch.from_numpy(facs[0]["sfc_albedo"]).to(dev)
            ka_all = torch.from_numpy(np.stack([f["k_abs"] for f in facs])).pin_memory()     # [112][nz]
            kr_all = torch.from_numpy(np.stack([f["k_ray"] for f in facs])).pin_memory()
            resident = None
        else:
            resident = [[make_optics_torch(cfg, p, device=dev)[k] for k in names] for p in pts]
        pinned_all = None
        # two contexts on two streams, points alternating, so that one point's pack and trace fill the SMs the
        # previous point's draining persistent kernel frees; the integer tallies of the two are summed
        from paper_2208_05247_b200.sweeps import spectral_sweep_batched
        batched = args.contexts == 0       # all points' optics in HBM slots, one launch (rt_trace_batch)
        if batched:
            g.set_slots(len(pts))
        extra = [rt.Grid(*cfg.grid, device=local, **cfg.accel) for _ in range(max(args.contexts, 1) - 1)]
        for gx in extra:
            gx.set_mode(weighted=(args.mode == "weighted"))
        sweep_streams = [torch.cuda.Stream(dev) for _ in range(max(args.contexts, 2))]
        pinned_cols2 = rt.Tallies(None, *[torch.empty((cfg.ny, cfg.nx), dtype=torch.int64).pin_memory()
                                          for _ in range(4)], counters=None)
    else:
        resident = [t.to(dev) for t in host]
        pinned_all = rt.Tallies(torch.empty((cfg.nz, cfg.ny, cfg.nx), dtype=torch.int64).pin_memory(),
                                pinned_cols.sfc_dir, pinned_cols.sfc_dif, pinned_cols.sfc_abs, pinned_cols.toa_up,
                                counters=None)
    point_ms = []

    def set_factored(kc, al, g=g):
        """All 112 points from their factors: kept factored in the trace (rt_set_cloud + rt_set_point; default) or
        packed into 16-byte records per voxel and point (rt_set_optics_factored; --packed-slots)."""
        if args.packed_slots:
            for j, f in enumerate(facs):
                g.set_optics_factored(j, kc, f["k_abs"], f["k_ray"], f["cloud_ssa"], f["cloud_g"], al)
        else:
            g.set_cloud(kc)
            if args.point_by_point:
                for j, f in enumerate(facs):
                    g.set_point(j, f["k_abs"], f["k_ray"], f["cloud_ssa"], f["cloud_g"], al)
            else:                          # rt_set_points: all 112 in one call (one albedo for all points)
                g.set_points(0, ka_all, kr_all, [f["cloud_ssa"] for f in facs], [f["cloud_g"] for f in facs], al)

    sweep_ms = []                      # spectral sweep: device time of set-up + trace per step
    def step(i, fields, out):
        g.reset_tallies()
        first = weak_range(rank, world, i, n)[0]
        if spectral:
            for gx in extra:
                gx.reset_tallies()
            ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ea.record()
            if batched and factored:
                set_factored(kc_dev, al_dev)                                        # S0, S1 from the factors
                g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, first_photon_id=first, seed=cfg.seed)
            elif batched:
                spectral_sweep_batched(g, lambda j: fields[j], counts, cfg.zenith_deg, cfg.azimuth_deg,
                                       seed=cfg.seed, first_photon_id=first)       # 112 x (S0, S1), one S2-S10 launch
            else:
                spectral_sweep_overlapped([g] + extra, sweep_streams, lambda j: fields[j], counts, cfg.zenith_deg,
                                          cfg.azimuth_deg, seed=cfg.seed, first_photon_id=first)   # 112 x (S0, S1, S2-S10)
            eb.record()
            t = g.read_tallies(out=out)                          # S11, both contexts
            for gx in extra:
                t2 = gx.read_tallies(out=pinned_cols2)
                for name in ("sfc_dir", "sfc_dif", "sfc_abs", "toa_up"):
                    getattr(t, name).add_(getattr(t2, name))
                for name, _ in rt.rt_counters._fields_:
                    setattr(t.counters, name, getattr(t.counters, name) + getattr(t2.counters, name))
            if t.counters.n_photons != n or t.counters.n_capped != 0:
                raise SystemExit("bench.py: photon count mismatch (%d of %d)" % (t.counters.n_photons, n))
            # one launch traces the whole sweep (batched): its own device time is the kernel's; the events around the
            # sweep also hold the set-up of the 112 points and the host's gaps between those calls
            sweep_ms.append(ea.elapsed_time(eb))
            return t, (g.last_trace_ms() if batched else sweep_ms[-1])
        else:
            g.set_optics(*fields)                                    # S0 pack, S1 majorant
            g.trace(cfg.zenith_deg, cfg.azimuth_deg, n, first_photon_id=first, seed=cfg.seed)  # S2-S10
            ms = None
        t = g.read_tallies(out=out)                              # S11
        if t.counters.n_photons != n or t.counters.n_capped != 0:
            raise SystemExit("bench.py: photon count mismatch (%d of %d, %d capped)" % (
                t.counters.n_photons, n, t.counters.n_capped))
        return t, (g.last_trace_ms() if ms is None else ms)

    for i in range(args.warmup):
        step(i, resident, pinned_cols)
    sweep_ms.clear()

    # ---- device-timed region: inputs resident in HBM ---------------------------------------------------
    uuid = None
    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
    except Exception:
        pass
    sampler = ClockSampler(uuid) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = g.launch_count() + (sum(gx.launch_count() for gx in extra) if spectral else 0)
    events = sfc_hits = 0
    csum = {}
    trace_ms = []
    barrier()
    e0.record()
    for i in range(args.steps):
        t, ms = step(args.warmup + i, resident, pinned_cols)
        events += t.counters.n_events
        sfc_hits += t.counters.n_sfc_hits
        for k, v in t.counters.asdict().items():
            csum[k] = csum.get(k, 0) + v
        trace_ms.append(ms)
    e1.record()
    barrier()
    elapsed_ms = max_over_ranks(e0.elapsed_time(e1))
    launches = g.launch_count() + (sum(gx.launch_count() for gx in extra) if spectral else 0) - launches0
    clocks = sampler.stop() if sampler else None
    closure_ok = (args.mode == "analog" and
                  int(t.sfc_abs.sum()) + int(t.toa_up.sum()) + t.counters.n_atm_abs * rt.W0 == n * rt.W0)
    if args.mode == "weighted":     # atm_abs stays on the device in this leg: sum it there
        ta = g.read_tallies(host=False)
        closure_ok = ta.closure() == n * rt.W0
        del ta

    total_photons = n * world * args.steps
    total_events = sum_over_ranks(events)
    value = total_photons / (elapsed_ms * 1e-3)

    # ---- the path's one exchange step, outside the timed region ---------------------------
    # One JOB of world x 2^22 photons split over the ranks by job index (rt_trace_range), then ONE exact int64
    # all-reduce of the device tallies over NCCL: the merged tallies must close to the job's energy and every
    # rank must hold the same sums.  (At world = 1 the same calls run without a collective.)
    exchange = None
    if not spectral:
        from paper_2208_05247_b200.shard import job_range, allreduce_tallies
        job = world * min(n, 1 << 22)
        begin, count = job_range(rank, world, job)
        g.reset_tallies()
        g.trace_range(cfg.zenith_deg, cfg.azimuth_deg, job, begin, count, first_photon_id=1 << 40, seed=cfg.seed)
        td = g.read_tallies(host=False)
        parts = [td.atm_abs, td.sfc_dir, td.sfc_dif, td.sfc_abs, td.toa_up]
        led = torch.tensor([td.counters.capped_energy + td.counters.roulette_lost - td.counters.roulette_gained,
                            td.counters.n_photons], dtype=torch.int64, device=dev)
        torch.cuda.synchronize(dev)
        x0 = time.perf_counter()
        allreduce_tallies(parts + [led])
        torch.cuda.synchronize(dev)
        x_ms = 1e3 * (time.perf_counter() - x0)
        merged = int(td.atm_abs.sum()) + int(td.sfc_abs.sum()) + int(td.toa_up.sum()) + int(led[0])
        ok = merged == job * rt.W0 and int(led[1]) == job
        if not ok:
            raise SystemExit("bench.py: all-reduced tallies do not close (%d of %d quanta)" % (merged, job * rt.W0))
        exchange = {"tallies_allreduced": world > 1, "ranks": world, "job_photons": job, "closure_exact": bool(ok),
                    "allreduce_bytes": sum(p.numel() * 8 for p in parts), "allreduce_ms": max_over_ranks(x_ms),
                    "how": "rt_trace_range per rank + one int64 sum all-reduce (NCCL) of atm_abs and the four column tallies"}
        del td, parts

    # ---- end-to-end leg: host fields in, all tallies out to the host, every step --------------------------
    # Two contexts on two streams, steps alternating: while one context traces, the other uploads its next fields
    # (pinned host memory, inside rt_set_optics) and downloads its last tallies (rt_read_tallies_async), so the
    # PCIe copies of every step are in the timed region but off the critical path.  Every step is checked after
    # the final synchronisation.  --e2e-serial keeps everything on one context and one stream.
    e2e = None
    if spectral and factored and batched:
        # spectral sweep end to end: the cloud field and the albedo come from pinned host memory every step, the
        # gas profiles (2 nz numbers per point) from plain host arrays, all tallies go back to the host
        import ctypes
        kc_host = torch.from_numpy(facs[0]["k_cloud"]).pin_memory()
        al_host = torch.from_numpy(facs[0]["sfc_albedo"]).pin_memory()
        out_all = rt.Tallies(torch.empty((cfg.nz, cfg.ny, cfg.nx), dtype=torch.int64).pin_memory(),
                             pinned_cols.sfc_dir, pinned_cols.sfc_dif, pinned_cols.sfc_abs, pinned_cols.toa_up,
                             counters=None)

        def e2e_sweep(i):
            g.reset_tallies()
            if args.packed_slots:
                kc_dev.copy_(kc_host, non_blocking=True)
                al_dev.copy_(al_host, non_blocking=True)
                set_factored(kc_dev, al_dev)
            else:
                set_factored(kc_host, al_host)           # the library copies the host fields itself
            g.trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts, first_photon_id=weak_range(rank, world, i, n)[0],
                          seed=cfg.seed)
            t = g.read_tallies(out=out_all)
            if t.counters.n_photons != n or t.counters.n_capped != 0:
                raise SystemExit("bench.py: e2e photon count mismatch (%d of %d)" % (t.counters.n_photons, n))

        if args.e2e_serial or args.packed_slots:
            e2e_sweep(0)
            barrier()
            t0 = time.perf_counter()
            for i in range(args.steps):
                e2e_sweep(args.warmup + args.steps + i)
            barrier()
            e2e_s = max_over_ranks(time.perf_counter() - t0)
            how = "one context, synchronous read"
        else:
            # as the e2e leg of the other workloads: sweeps alternate over two contexts on two streams, so that one
            # sweep's uploads and read-out overlap the other's trace
            g2 = rt.Grid(*cfg.grid, device=local, **cfg.accel)
            g2.set_mode(weighted=(args.mode == "weighted"))
            g2.set_slots(len(pts))
            ctxs, streams2 = [g, g2], [torch.cuda.Stream(dev), torch.cuda.Stream(dev)]
            outs = [out_all, rt.Tallies(torch.empty((cfg.nz, cfg.ny, cfg.nx), dtype=torch.int64).pin_memory(),
                                        *[torch.empty((cfg.ny, cfg.nx), dtype=torch.int64).pin_memory() for _ in range(4)],
                                        counters=None)]
            cbufs = [torch.zeros(ctypes.sizeof(rt.rt_counters), dtype=torch.uint8).pin_memory() for _ in range(2)]

            def e2e_start(i, k):
                with torch.cuda.stream(streams2[k]):
                    set_factored(kc_host, al_host, ctxs[k])     # uploads first: they overlap the other context's trace
                    ctxs[k].reset_tallies()
                    ctxs[k].trace_batch(cfg.zenith_deg, cfg.azimuth_deg, counts,
                                        first_photon_id=weak_range(rank, world, i, n)[0], seed=cfg.seed)
                    ctxs[k].read_tallies_async(outs[k], cbufs[k])

            def e2e_finish(k):
                streams2[k].synchronize()
                cnt = rt.counters_of(cbufs[k])
                if cnt.n_photons != n or cnt.n_capped != 0:
                    raise SystemExit("bench.py: e2e photon count mismatch (%d of %d)" % (cnt.n_photons, n))

            for k in range(2):
                e2e_start(k, k)
            for k in range(2):
                e2e_finish(k)
            barrier()
            t0 = time.perf_counter()
            for i in range(args.steps):
                k = i & 1
                if i >= 2:
                    e2e_finish(k)
                e2e_start(args.warmup + args.steps + i, k)
            for k in range(2):
                e2e_finish(k)
            barrier()
            e2e_s = max_over_ranks(time.perf_counter() - t0)
            how = "two contexts on two streams, sweeps alternating; copies overlap the other context's trace"
            g2.close()
        h2d = kc_host.numel() * 4 + al_host.numel() * 4 + len(facs) * 2 * cfg.nz * 4
        d2h = (cfg.nvox + 4 * cfg.ncol) * 8 + ctypes.sizeof(rt.rt_counters)
        e2e = {"value": total_photons / e2e_s, "unit": UNIT, "ms_per_step": 1e3 * e2e_s / args.steps,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "how": "factored inputs: cloud field + albedo from pinned host memory, 112 x 2 nz profile values; "
                      "all tallies to pinned host memory; " + how}
    if not spectral:
        import ctypes
        h2d = sum(x.numel() * x.element_size() for x in host)
        d2h = (cfg.nvox + 4 * cfg.ncol) * 8 + ctypes.sizeof(rt.rt_counters)
        if args.e2e_serial:
            step(0, host, pinned_all)
            barrier()
            t0 = time.perf_counter()
            for i in range(args.steps):
                step(args.warmup + args.steps + i, host, pinned_all)
            barrier()
            e2e_s = max_over_ranks(time.perf_counter() - t0)
            how = "one context, synchronous copies"
        else:
            ctxs = [g, rt.Grid(*cfg.grid, device=local, **cfg.accel)]
            ctxs[1].set_mode(weighted=(args.mode == "weighted"))
            streams2 = [torch.cuda.Stream(dev), torch.cuda.Stream(dev)]
            outs = [pinned_all, rt.Tallies(torch.empty((cfg.nz, cfg.ny, cfg.nx), dtype=torch.int64).pin_memory(),
                                           *[torch.empty((cfg.ny, cfg.nx), dtype=torch.int64).pin_memory() for _ in range(4)],
                                           counters=None)]
            cbufs = [torch.zeros(ctypes.sizeof(rt.rt_counters), dtype=torch.uint8).pin_memory() for _ in range(2)]

            def e2e_step(i, k):
                with torch.cuda.stream(streams2[k]):
                    ctxs[k].set_optics(*host)      # H2D copies first: they overlap the other context's trace
                    ctxs[k].reset_tallies()        # (a memset needs SMs and would wait for that trace to drain)
                    ctxs[k].trace(cfg.zenith_deg, cfg.azimuth_deg, n, first_photon_id=weak_range(rank, world, i, n)[0],
                                  seed=cfg.seed)
                    ctxs[k].read_tallies_async(outs[k], cbufs[k])

            def e2e_check(k):
                streams2[k].synchronize()
                cnt = rt.counters_of(cbufs[k])
                if cnt.n_photons != n or cnt.n_capped != 0:
                    raise SystemExit("bench.py: e2e photon count mismatch (%d of %d)" % (cnt.n_photons, n))

            for k in range(2):
                e2e_step(k, k)
            for k in range(2):
                e2e_check(k)
            barrier()
            t0 = time.perf_counter()
            for i in range(args.steps):
                k = i & 1
                if i >= 2:
                    e2e_check(k)                 # the step that used these buffers two steps ago
                e2e_step(args.warmup + args.steps + i, k)
            for k in range(2):
                e2e_check(k)
            barrier()
            e2e_s = max_over_ranks(time.perf_counter() - t0)
            how = "two contexts on two streams, steps alternating; copies overlap the other context's trace"
            ctxs[1].close()
        e2e = {"value": total_photons / e2e_s, "unit": UNIT, "ms_per_step": 1e3 * e2e_s / args.steps,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "how": how}

    # ---- roofline of the dominant kernel (trace_kernel), this rank ---------------------------------------
    # the path's bound is the memory GATHER rate.  Two ceilings are measured in this run by
    # rt_gather_bench (8 independent random 16 B loads in flight per thread = one 32 B sector each): over the whole
    # packed-optics array (HBM) and over its first 16 MiB (L2).  The time a perfect kernel would need for THIS
    # launch's memory work is max(L2 read sectors / L2 gather rate, DRAM read sectors / HBM gather rate), with the
    # sector counts of the shipped kernel from the committed ncu capture (profiles/trace_kernel_counters.json,
    # keyed by the kernel sources' hash); frac = that time / the kernel's measured time = achieved events/s over
    # the events/s the ceiling allows.  Without a capture of the kernel as it stands, the algorithmic model of
    # §8(d) is used: one 32 B sector from HBM per tentative collision.
    hbm_peak, peak_src = _peaks()
    ms_avg = sum(trace_ms) / len(trace_ms)
    per = {k: v / args.steps for k, v in csum.items()}
    ev_per_launch = per["n_events"]
    atomics_per_launch = n + per["n_sfc_hits"]
    alg_bytes = SECTOR * ev_per_launch + 2 * SECTOR * atomics_per_launch
    trace_events_per_s = ev_per_launch / (ms_avg * 1e-3)
    trace_gathers_per_s = (per["n_cell_steps"] + 2 * per["n_events"]) / (ms_avg * 1e-3)   # majorant + voxel loads
    gather = {}
    for label, foot in (("hbm_whole_array", 0), ("l2_16MiB", min(1 << 20, cfg.nvox))):
        gb_ms, gb_loads = g.gather_bench(64, foot)
        gather[label] = gb_loads / (gb_ms * 1e-3)
    ncu = _ncu_counters(cfg, args.mode, n) if (not spectral or (args.contexts == 0 and not args.packed_slots and not args.full_fields)) else None
    if ncu:
        # sector counts for the roof: where the shipped build spills registers (the 5-blocks-per-SM instantiations), those
        # of the same sources built without spills (profiles/trace_kernel_counters.md): reloading spilled registers is
        # not work a perfect kernel would do, and counting it would RAISE the fraction
        roof_l2 = ncu.get("roof_lts_t_sectors_op_read", ncu["lts_t_sectors_op_read"])
        roof_dram = ncu.get("roof_dram_bytes_read", ncu["dram_bytes_read"])
        t_l2 = roof_l2 / gather["l2_16MiB"]
        t_hbm = roof_dram / SECTOR / gather["hbm_whole_array"]
        t_hbm_stream = (roof_dram + ncu["dram_bytes_write"]) / (hbm_peak * 1e9)
        hbm_term = "gather"
        if t_hbm > ms_avg * 1e-3:
            # the kernel moved its DRAM sectors FASTER than the microbenchmark gathers uniformly random ones (config 5:
            # its misses on the majorant table have row locality), so that rate is no ceiling for this launch; what
            # remains a bound is the same traffic at the streaming rate ("if locality lets the tracer
            # beat the uniform-random HBM ceiling ...")
            t_hbm, hbm_term = t_hbm_stream, "stream"
        t_roof = max(t_l2, t_hbm)
        traffic = ncu["dram_bytes_read"] + ncu["dram_bytes_write"]
        model = ("max(L2 read sectors / L2 gather rate, DRAM read sectors / HBM gather rate); sector counts from "
                 "profiles/trace_kernel_counters.json (kernel_sha16 %s), gather rates measured in this run" % ncu["kernel_sha16"])
        sm_mhz = _sm_max_mhz()
        lane_peak = 148 * 4 * 32 * sm_mhz * 1e6
        alu = {"thread_inst_per_launch": ncu["thread_inst_executed"], "warp_inst_per_launch": ncu["inst_executed"],
               "active_lanes_per_inst": ncu["thread_inst_executed"] / ncu["inst_executed"],
               "issue_active_pct_ncu": ncu["issue_active_pct"],
               "lane_slots_used": ncu["thread_inst_executed"] / (ms_avg * 1e-3) / lane_peak,
               "issue_slots_used": ncu["inst_executed"] / (ms_avg * 1e-3) / (148 * 4 * sm_mhz * 1e6),
               "peak": "148 SMs x 4 sub-partitions x 32 lanes x %.0f MHz; instruction counts measured by ncu" % sm_mhz}
    else:
        t_l2, t_hbm = None, ev_per_launch / gather["hbm_whole_array"]
        t_hbm_stream, hbm_term = None, "gather"
        t_roof = t_hbm
        traffic = None
        alu = None
        model = ("no ncu capture of the kernel as it stands: SURVEY.md 8(d)'s algorithmic model, one 32 B sector from "
                 "HBM per tentative collision")
    roof_events_per_s = ev_per_launch / t_roof

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle as O
        cores = O.hardware_threads()
        ot, _, el = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, CPU_BASELINE_PHOTONS, seed=cfg.seed,
                            precision=64, n_threads=cores, weighted=(args.mode == "weighted"), **cfg.accel)
        cpu = {"value": CPU_BASELINE_PHOTONS / el, "unit": UNIT, "cores": cores, "kind": "oracle",
               "collision_events_per_s": ot.counters.n_events / el,
               "sample": "photon ids [0, %d) (%d per column) of the %d-photon workload, photon loop only" % (
                   CPU_BASELINE_PHOTONS, CPU_BASELINE_PHOTONS // cfg.ncol, n)}

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "collision_events_per_s": total_events / (elapsed_ms * 1e-3),
        "events_per_photon": total_events / total_photons,
        "per_photon": {k: per[k] / n for k in ("n_events", "n_null", "n_hg", "n_rayleigh", "n_cell_steps", "n_relevel",
                                               "n_sfc_hits")},
        "spectral_sweep": ({"device_ms": sum(sweep_ms) / len(sweep_ms), "trace_ms": ms_avg,
                            "set_up_ms": sum(sweep_ms) / len(sweep_ms) - ms_avg} if sweep_ms else None),
        "trace_kernel": {"ms": ms_avg, "paths_per_s": n / (ms_avg * 1e-3), "events_per_s": trace_events_per_s},
        "config": {"workload": cfg.name, "grid": [cfg.nx, cfg.ny, cfg.nz], "photons_per_gpu_per_step": n,
                   "block": list(cfg.block), "merge": list(cfg.merge), "merge_ratio": cfg.merge_ratio,
                   "mode": args.mode, "factored_inputs": bool(spectral and not args.full_fields and args.contexts == 0),
                   "zenith_deg": cfg.zenith_deg, "azimuth_deg": cfg.azimuth_deg,
                   "parallelism": "photon-id ranges per GPU, no collective" if world > 1 else "1 GPU",
                   "l2": ("inputs exceed L2 (%d MiB packed optics + %d MiB tallies vs 126 MB)" % (
                       cfg.nvox * 16 >> 20, cfg.nvox * 8 >> 20)) if cfg.nvox * 24 > (126 << 20) else
                         "inputs fit L2; every step traces new photon ids",
                   "step": ("reset_tallies + set_cloud + set_points for the 112 points (--point-by-point: 112 x set_point; --packed-slots: 112 x set_optics_factored; "
                            "--full-fields: 112 x set_optics_slot) + one trace_batch launch (stream_id = point) + "
                            "read_tallies" if spectral and args.contexts == 0 else
                            "reset_tallies + 112 x (set_optics + trace, stream_id = point; points alternating over "
                            "--contexts contexts and streams) + read_tallies of all"
                            if spectral else
                            "reset_tallies + set_optics + trace + read_tallies(column tallies, counters)")},
        "e2e": e2e,
        "gpu_launches": launches,
        "closure_exact": bool(closure_ok),
        "clocks": clocks,
        "roofline": {"bound": "gather", "achieved": trace_events_per_s, "peak": roof_events_per_s,
                     "unit": "tentative collisions/s", "frac": trace_events_per_s / roof_events_per_s,
                     "traffic": traffic, "kernel": "trace_kernel", "model": model,
                     "events_per_launch": ev_per_launch, "kernel_ms": ms_avg,
                     "roof_ms": 1e3 * t_roof, "roof_ms_l2": None if t_l2 is None else 1e3 * t_l2, "roof_ms_hbm": 1e3 * t_hbm,
                     "roof_hbm_term": hbm_term + (" (DRAM bytes at the streaming copy rate: the launch beat the uniform-random gather rate, "
                                                  "which would give %.1f ms)" % (1e3 * roof_dram / SECTOR / gather["hbm_whole_array"])
                                                  if hbm_term == "stream" else " (DRAM read sectors at the measured random-gather rate)"),
                     "roof_ms_hbm_stream": None if t_hbm_stream is None else 1e3 * t_hbm_stream,
                     "gather_sectors_per_s": gather,
                     "frac_events_vs_hbm_gather": trace_events_per_s / gather["hbm_whole_array"],
                     "frac_all_gathers_vs_l2_gather": trace_gathers_per_s / gather["l2_16MiB"],
                     "ncu": ncu},
        "alu": alu,
        "hbm": {"algorithmic_GBps": alg_bytes / (ms_avg * 1e-3) / 1e9, "peak_GBps": hbm_peak, "peak_source": peak_src,
                "frac": alg_bytes / (ms_avg * 1e-3) / 1e9 / hbm_peak,
                "bytes_model": "32 B sector per tentative collision + 2 x 32 B per tally atomic (SURVEY.md 8(d)), "
                               "against the streaming copy rate: context only, a random gather cannot reach it"},
        "exchange": exchange,
        "cpu_baseline": cpu,
    }))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--workload", type=int, choices=(1, 2, 3, 4, 5), default=WORKLOAD,
                    help="BASELINE.json configs[N-1]; the default (3) is the configuration the metric is quoted on")
    ap.add_argument("--point-by-point", action="store_true",
                    help="workload 4: one rt_set_point call per spectral point instead of one rt_set_points call")
    ap.add_argument("--block", default=None, help="acceleration-grid block bx,by,bz (default: the config's)")
    ap.add_argument("--mode", choices=("analog", "weighted"), default="analog",
                    help="absorption scheme: analog (the metric's, default) or the paper's weights + roulette")
    ap.add_argument("--contexts", type=int, default=0,
                    help="workload 4: 0 (default) = all points' optics in HBM slots and one launch (rt_trace_batch); "
                         "N >= 1 = one rt_trace per point, points alternating over N contexts on N streams")
    ap.add_argument("--merge", default=None, help="merged-cell factors mx,my,mz (default: the config's; 1,1,1 = off)")
    ap.add_argument("--packed-slots", action="store_true",
                    help="workload 4 with factored inputs: pack a 16-byte record per voxel and point "
                         "(rt_set_optics_factored) instead of keeping the optics factored in the trace "
                         "(rt_set_cloud + rt_set_point, the default)")
    ap.add_argument("--full-fields", action="store_true",
                    help="workload 4: give every point's optics as four full 3-D fields (rt_set_optics_slot) instead of "
                         "as factors (one cloud field + per-level gas profiles per point, rt_set_optics_factored)")
    ap.add_argument("--e2e-serial", action="store_true", help="e2e leg on one context with synchronous copies")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing (used under ncu)")
    args = ap.parse_args()
    if args.steps < 1 or args.warmup < 0:
        raise SystemExit("bench.py: --steps >= 1, --warmup >= 0")
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
