"""Host loops over the C-ABI calls for the two multi-call workloads of BASELINE.json: the spectral sweep
(configs[3]: 112 independent spectral points on one field, "for each spectral quadrature
point") and the convergence sweep (configs[4]: 1-256 photons per surface column).  Argument
marshalling only: every step of the path runs in the kernels behind rt_set_optics / rt_trace."""
import torch


def spectral_sweep(grid, fields_of_point, counts, zenith_deg, azimuth_deg, seed=1, first_photon_id=0,
                   timings=None):
    """Trace point j with counts[j] photons on stream_id = j, tallies accumulated in `grid` (equal power per
    photon, so the sums are broadband).  `fields_of_point(j)` returns the five rt_set_optics
    arrays of point j (device or host).  Everything is queued on the current stream; returns the photon total.
    `timings` (a list) receives (j, trace ms) per point; reading it makes each point synchronise."""
    total = 0
    for j, n in enumerate(counts):
        if n == 0:
            continue
        grid.set_optics(*fields_of_point(j))
        grid.trace(zenith_deg, azimuth_deg, n, first_photon_id=first_photon_id, seed=seed, stream_id=j)
        if timings is not None:
            timings.append((j, grid.last_trace_ms()))
        total += n
    return total


def spectral_sweep_overlapped(grids, streams, fields_of_point, counts, zenith_deg, azimuth_deg, seed=1,
                              first_photon_id=0):
    """The same sweep over several contexts of the same grid (normally two), point j going to context j mod
    len(grids) on that context's own stream: while the persistent trace kernel of one point drains (a point
    of config 4 is only ~6e5 photons, so its tail is a large part of its launch), the next point's pack and
    trace already fill the freed SMs.  Each context accumulates its own tallies; their sum (exact, int64) is
    the sweep's result: `sum_tallies`.  The streams wait for the caller's current stream first."""
    ready = torch.cuda.Event()
    ready.record()
    for st in streams:
        st.wait_event(ready)
    total = 0
    k = 0
    for j, n in enumerate(counts):
        if n == 0:
            continue
        g, st = grids[k % len(grids)], streams[k % len(grids)]
        k += 1
        with torch.cuda.stream(st):
            g.set_optics(*fields_of_point(j))
            g.trace(zenith_deg, azimuth_deg, n, first_photon_id=first_photon_id, seed=seed, stream_id=j)
        total += n
    for st in streams:
        torch.cuda.current_stream().wait_stream(st)
    return total


def spectral_sweep_batched(grid, fields_of_point, counts, zenith_deg, azimuth_deg, seed=1, first_photon_id=0):
    """The same sweep with every point's packed optics resident in its own HBM slot (`grid.set_slots(len(counts))`
    beforehand; 16 B per voxel and point: 57 GB for config 4) and ONE launch for all points (rt_trace_batch):
    no launch drains between points and the host waits once, not once per point.  Traces exactly the photons of
    spectral_sweep (same ids, stream ids, column stratification), so the integer tallies are identical."""
    for j in range(len(counts)):
        grid.set_optics_slot(j, *fields_of_point(j))
    grid.trace_batch(zenith_deg, azimuth_deg, counts, first_photon_id=first_photon_id, seed=seed)
    return sum(int(x) for x in counts)


def sum_tallies(grids, host=False):
    """Sum of the contexts' tallies and counters (integers: exact and order-independent)."""
    from .binding import Tallies, rt_counters
    ts = [g.read_tallies(host=host) for g in grids]
    cnt = rt_counters()
    for name, _ in rt_counters._fields_:
        setattr(cnt, name, sum(int(getattr(t.counters, name)) for t in ts))
    fields = [sum(getattr(t, f) for t in ts[1:]) + getattr(ts[0], f) if len(ts) > 1 else getattr(ts[0], f)
              for f in ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up")]
    return Tallies(*fields, counters=cnt)


def _block_sums(t, blk):
    """Sums over blocks of blk voxels/columns of an integer tensor whose shape is a multiple of blk."""
    shp = []
    for n, b in zip(t.shape, blk):
        shp += [n // b, b]
    return t.reshape(shp).sum(dim=tuple(range(1, 2 * len(blk), 2)))


def convergence_sweep(grid, ncol, per_column, zenith_deg, azimuth_deg, seed=1, reference_per_column=256,
                      sfc_block=(16, 16), vox_block=(16, 32, 32), min_hits=500):
    """RMS relative noise of surface irradiance and voxel heating against the photons per column.
    A reference launch of reference_per_column photons per column on ids disjoint from every test launch;
    then one launch per entry of per_column from id 0.  Noise = RMS over blocks (sfc_block columns,
    vox_block voxels as (z, y, x)) with >= min_hits reference hits of (T_N / N - R / N_ref) / (R / N_ref), so
    its expectation is c sqrt(1/N + 1/N_ref).  Returns one dict per entry with the launch's device time."""
    n_ref = reference_per_column * ncol
    grid.reset_tallies()
    grid.trace(zenith_deg, azimuth_deg, n_ref, first_photon_id=1 << 40, seed=seed)
    ref = grid.read_tallies(host=False)
    ref_ms = grid.last_trace_ms()
    r_sfc = _block_sums(ref.sfc_dir + ref.sfc_dif, sfc_block).double()
    r_abs = _block_sums(ref.atm_abs, vox_block).double()
    m_sfc = r_sfc >= min_hits * float(1 << 32)
    m_abs = r_abs >= min_hits * float(1 << 32)
    del ref
    out = []
    for ppc in per_column:
        n = ppc * ncol
        grid.reset_tallies()
        grid.trace(zenith_deg, azimuth_deg, n, first_photon_id=0, seed=seed)
        t = grid.read_tallies(host=False)
        ms = grid.last_trace_ms()
        scale = reference_per_column / ppc
        s = _block_sums(t.sfc_dir + t.sfc_dif, sfc_block).double() * scale
        a = _block_sums(t.atm_abs, vox_block).double() * scale
        rel_s = ((s - r_sfc) / r_sfc)[m_sfc]
        rel_a = ((a - r_abs) / r_abs)[m_abs]
        out.append({"photons_per_column": ppc, "n_photons": n, "trace_ms": ms,
                    "paths_per_s": n / (ms * 1e-3),
                    "closure_exact": bool(int(t.atm_abs.sum()) + int(t.sfc_abs.sum()) + int(t.toa_up.sum())
                                          + int(t.counters.capped_energy) == n << 32),
                    "n_events": t.counters.n_events, "n_capped": t.counters.n_capped,
                    "rms_noise_sfc": float(torch.sqrt((rel_s ** 2).mean())), "sfc_blocks": int(m_sfc.sum()),
                    "rms_noise_heating": float(torch.sqrt((rel_a ** 2).mean())), "heating_blocks": int(m_abs.sum())})
        del t, s, a
    return out, {"photons_per_column": reference_per_column, "n_photons": n_ref, "trace_ms": ref_ms}
