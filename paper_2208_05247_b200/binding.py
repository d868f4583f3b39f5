"""Thin ctypes binding of include/rt.h (librt_b200.so).  Argument marshalling only: every step of
the method runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.
There is no CPU fallback: a missing library or a failed call raises."""
import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "librt_b200.so")
W0 = 1 << 32
FATE_ATM_ABS, FATE_SFC_ABS, FATE_TOD_EXIT, FATE_CAPPED, FATE_ROULETTE = 1, 2, 3, 4, 5
MODE_ANALOG, MODE_WEIGHTED = 0, 1

EXPORTS = ("rt_create_grid", "rt_set_merge", "rt_set_mode", "rt_set_source", "rt_set_optics", "rt_set_slots", "rt_set_optics_slot", "rt_set_optics_factored", "rt_set_cloud", "rt_set_point", "rt_set_points", "rt_trace_batch", "rt_trace", "rt_trace_records", "rt_trace_range", "rt_read_tallies", "rt_read_tallies_async",
           "rt_reset_tallies", "rt_set_heating_split", "rt_read_heating_direct", "rt_tally_to_flux", "rt_read_majorant", "rt_read_packed_optics", "rt_gather_bench",
           "rt_last_trace_ms", "rt_launch_count", "rt_philox_words", "rt_selftest_ieee", "rt_majorant_no_alloc", "rt_no_alloc_last_error", "rt_last_error", "rt_destroy")

COUNTER_FIELDS = ("n_photons", "n_events", "n_null", "n_rayleigh", "n_hg", "n_atm_abs", "n_sfc_hits",
                  "n_sfc_abs", "n_toa", "n_capped", "n_cell_steps", "n_relevel", "n_roulette_killed", "n_roulette_kept",
                  "capped_energy", "roulette_lost", "roulette_gained")
N_SIGNED = 3


class RtError(RuntimeError):
    pass


class rt_counters(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in COUNTER_FIELDS[:-N_SIGNED]] + [(n, C.c_int64) for n in COUNTER_FIELDS[-N_SIGNED:]]

    def asdict(self):
        return {n: int(getattr(self, n)) for n in COUNTER_FIELDS}


_lib = None


def lib():
    """Load librt_b200.so (built by paper_2208_05247_b200.build); raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RtError("CUDA library %s is missing: run `python -m paper_2208_05247_b200.build` "
                      "(there is no CPU fallback)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, i32, u32, u64, f32, f64 = C.c_void_p, C.c_int, C.c_uint32, C.c_uint64, C.c_float, C.c_double
    L.rt_create_grid.argtypes = [C.POINTER(vp), i32, i32, i32, f32, f32, f32, i32, i32, i32, i32]
    L.rt_set_merge.argtypes = [vp, i32, i32, i32, f32]
    L.rt_set_mode.argtypes = [vp, i32]
    L.rt_set_source.argtypes = [vp, f32, i32]
    L.rt_set_optics.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    L.rt_set_slots.argtypes = [vp, i32]
    L.rt_set_optics_slot.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
    L.rt_set_optics_factored.argtypes = [vp, i32, vp, vp, vp, f32, f32, vp, vp]
    L.rt_set_cloud.argtypes = [vp, vp, vp]
    L.rt_set_point.argtypes = [vp, i32, vp, vp, f32, f32, vp, vp]
    L.rt_set_points.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, u64, vp]
    L.rt_trace_batch.argtypes = [vp, f64, f64, i32, i32, C.POINTER(u64), u64, u64, vp, vp]
    L.rt_trace.argtypes = [vp, f64, f64, u64, u64, u64, u32, vp]
    L.rt_trace_records.argtypes = [vp, f64, f64, u64, u64, u64, u32, vp, vp]
    L.rt_trace_range.argtypes = [vp, f64, f64, u64, u64, u64, u32, vp, u64, u64, vp]
    L.rt_read_tallies.argtypes = [vp, vp, vp, vp, vp, vp, C.POINTER(rt_counters)]
    L.rt_read_tallies_async.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
    L.rt_reset_tallies.argtypes = [vp, vp]
    L.rt_set_heating_split.argtypes = [vp, i32]
    L.rt_read_heating_direct.argtypes = [vp, vp]
    L.rt_tally_to_flux.argtypes = [vp, vp, u64, u64, u64, f64, f64]
    L.rt_read_majorant.argtypes = [vp, vp]
    L.rt_read_packed_optics.argtypes = [vp, vp]
    L.rt_gather_bench.argtypes = [vp, u32, u64, vp, C.POINTER(f32), C.POINTER(u64)]
    L.rt_last_trace_ms.argtypes = [vp, C.POINTER(f32)]
    L.rt_launch_count.argtypes = [vp]
    L.rt_launch_count.restype = u64
    L.rt_philox_words.argtypes = [i32, vp, u32, u32, vp, u64]
    L.rt_selftest_ieee.argtypes = [i32, C.POINTER(u64), C.POINTER(u64)]
    L.rt_majorant_no_alloc.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, i32, i32, i32, i32, f32, i32, vp]
    L.rt_no_alloc_last_error.argtypes = []
    L.rt_no_alloc_last_error.restype = C.c_char_p
    L.rt_last_error.argtypes = [vp]
    L.rt_last_error.restype = C.c_char_p
    L.rt_destroy.argtypes = [vp]
    L.rt_destroy.restype = None
    for name in EXPORTS:
        if name not in ("rt_launch_count", "rt_last_error", "rt_no_alloc_last_error", "rt_destroy"):
            getattr(L, name).restype = i32
    _lib = L
    return L


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(None)


def _stream(device):
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


class Tallies:
    """Tallies copied out by rt_read_tallies (torch int64, on the device or pinned host memory)."""

    def __init__(self, atm_abs, sfc_dir, sfc_dif, sfc_abs, toa_up, counters):
        self.atm_abs, self.sfc_dir, self.sfc_dif, self.sfc_abs, self.toa_up = atm_abs, sfc_dir, sfc_dif, sfc_abs, toa_up
        self.counters = counters

    def closure(self):
        return (int(self.atm_abs.sum()) + int(self.sfc_abs.sum()) + int(self.toa_up.sum())
                + int(self.counters.capped_energy) + int(self.counters.roulette_lost)
                - int(self.counters.roulette_gained))


def counters_of(buf):
    """rt_counters from the pinned byte buffer filled by Grid.read_tallies_async (after a stream sync)."""
    return rt_counters.from_buffer_copy(bytes(buf.cpu().numpy().tobytes()))


def tally_to_flux(tally, n_photons, ncol, tod_flux, depth=0.0):
    """rt_tally_to_flux on a host int64 tensor: W m^-2 per column (depth = 0) or W m^-3 (depth = dz)."""
    t = tally.contiguous()
    if t.is_cuda or t.dtype != torch.int64:
        raise RtError("tally_to_flux: a host int64 tensor (as rt_read_tallies returns) is required")
    out = torch.empty(t.shape, dtype=torch.float64)
    rc = lib().rt_tally_to_flux(_ptr(t), _ptr(out), t.numel(), int(n_photons), int(ncol), float(tod_flux), float(depth))
    if rc != 0:
        raise RtError("rt_tally_to_flux failed (%d)" % rc)
    return out


class Grid:
    """One rt_ctx: rt_create_grid / rt_set_optics / rt_trace / rt_read_tallies (include/rt.h)."""

    def __init__(self, nx, ny, nz, dx, dy, dz, bx=8, by=8, bz=8, device=0, merge=(1, 1, 1), merge_ratio=1.25):
        if not torch.cuda.is_available():
            raise RtError("no CUDA device: this library has no CPU path")
        self.L = lib()
        self.shape = (nz, ny, nx)
        self.block = (bx, by, bz)
        self.device = torch.device("cuda", device)
        self.ctx = C.c_void_p(None)
        rc = self.L.rt_create_grid(C.byref(self.ctx), nx, ny, nz, dx, dy, dz, bx, by, bz, device)
        if rc != 0:
            msg = self.L.rt_last_error(self.ctx).decode() if self.ctx else "bad arguments"
            if self.ctx:
                self.L.rt_destroy(self.ctx)
                self.ctx = C.c_void_p(None)
            raise RtError("rt_create_grid failed (%d): %s" % (rc, msg))
        if tuple(merge) != (1, 1, 1):
            self.set_merge(*merge, merge_ratio=merge_ratio)

    def set_merge(self, mx, my, mz, merge_ratio=1.25):
        """Merged acceleration cells (include/rt.h rt_set_merge); call before set_optics."""
        self._check(self.L.rt_set_merge(self.ctx, int(mx), int(my), int(mz), float(merge_ratio)), "rt_set_merge")

    def _check(self, rc, name):
        if rc != 0:
            raise RtError("%s failed (%d): %s" % (name, rc, self.L.rt_last_error(self.ctx).decode()))

    def _f32(self, a, n):
        """fp32 contiguous tensor on this device or on the host (the library copies host fields itself)."""
        t = torch.as_tensor(a)
        if t.is_cuda and t.device != self.device:
            t = t.to(self.device)
        if t.dtype != torch.float32 or not t.is_contiguous():
            t = t.to(dtype=torch.float32).contiguous()
        if t.numel() != n:
            raise RtError("field has %d elements, expected %d" % (t.numel(), n))
        return t

    def set_mode(self, weighted):
        """Absorption scheme of the following traces: analog (False) or the paper's weights + roulette (True)."""
        self._check(self.L.rt_set_mode(self.ctx, MODE_WEIGHTED if weighted else MODE_ANALOG), "rt_set_mode")

    def set_source(self, diffuse_fraction=0.0, sobol=False):
        """Top-of-domain source of the following traces (include/rt.h rt_set_source)."""
        self._check(self.L.rt_set_source(self.ctx, float(diffuse_fraction), 1 if sobol else 0), "rt_set_source")

    def set_optics(self, k_ext, k_ext_cloud, ssa, g, sfc_albedo):
        nz, ny, nx = self.shape
        nvox, ncol = nx * ny * nz, nx * ny
        ts = [self._f32(k_ext, nvox), self._f32(k_ext_cloud, nvox), self._f32(ssa, nvox),
              self._f32(g, nvox), self._f32(sfc_albedo, ncol)]
        self._check(self.L.rt_set_optics(self.ctx, *[_ptr(t) for t in ts], _stream(self.device)), "rt_set_optics")

    def set_slots(self, n_slots):
        """Optics / majorant / albedo slots for batched spectral points (include/rt.h rt_set_slots)."""
        self._check(self.L.rt_set_slots(self.ctx, int(n_slots)), "rt_set_slots")

    def set_optics_slot(self, slot, k_ext, k_ext_cloud, ssa, g, sfc_albedo):
        nz, ny, nx = self.shape
        nvox, ncol = nx * ny * nz, nx * ny
        ts = [self._f32(k_ext, nvox), self._f32(k_ext_cloud, nvox), self._f32(ssa, nvox),
              self._f32(g, nvox), self._f32(sfc_albedo, ncol)]
        self._check(self.L.rt_set_optics_slot(self.ctx, int(slot), *[_ptr(t) for t in ts], _stream(self.device)),
                    "rt_set_optics_slot")

    def set_optics_factored(self, slot, k_cloud, k_abs, k_ray, cloud_ssa, cloud_g, sfc_albedo):
        """include/rt.h rt_set_optics_factored: cloud field and albedo on the device, gas profiles (nz) anywhere."""
        nz, ny, nx = self.shape
        kc, al = self._f32(k_cloud, nx * ny * nz), self._f32(sfc_albedo, nx * ny)
        ka, kr = self._f32(k_abs, nz), self._f32(k_ray, nz)
        self._check(self.L.rt_set_optics_factored(self.ctx, int(slot), _ptr(kc), _ptr(ka), _ptr(kr), float(cloud_ssa),
                                                  float(cloud_g), _ptr(al), _stream(self.device)),
                    "rt_set_optics_factored")

    def set_cloud(self, k_cloud):
        """include/rt.h rt_set_cloud: the cloud extinction field shared by all spectral points."""
        nz, ny, nx = self.shape
        self._check(self.L.rt_set_cloud(self.ctx, _ptr(self._f32(k_cloud, nx * ny * nz)), _stream(self.device)),
                    "rt_set_cloud")

    def set_point(self, slot, k_abs, k_ray, cloud_ssa, cloud_g, sfc_albedo):
        """include/rt.h rt_set_point: a spectral point by its factors, kept factored in the trace."""
        nz, ny, nx = self.shape
        ka, kr, al = self._f32(k_abs, nz), self._f32(k_ray, nz), self._f32(sfc_albedo, nx * ny)
        self._check(self.L.rt_set_point(self.ctx, int(slot), _ptr(ka), _ptr(kr), float(cloud_ssa), float(cloud_g),
                                        _ptr(al), _stream(self.device)), "rt_set_point")

    def set_points(self, first_slot, k_abs, k_ray, cloud_ssa, cloud_g, sfc_albedo):
        """include/rt.h rt_set_points: len(cloud_ssa) consecutive slots in one call.  k_abs, k_ray: [n][nz];
        sfc_albedo: ncol values (one albedo for all points) or [n][ncol]."""
        nz, ny, nx = self.shape
        n = len(cloud_ssa)
        ka, kr = self._f32(k_abs, n * nz), self._f32(k_ray, n * nz)
        al = torch.as_tensor(sfc_albedo)
        shared = al.numel() == nx * ny
        al = self._f32(al, nx * ny * (1 if shared else n))
        ssa = (C.c_float * n)(*[float(x) for x in cloud_ssa])
        cg = (C.c_float * n)(*[float(x) for x in cloud_g])
        self._check(self.L.rt_set_points(self.ctx, int(first_slot), n, _ptr(ka), _ptr(kr), ssa, cg, _ptr(al),
                                         0 if shared else nx * ny, _stream(self.device)), "rt_set_points")

    def trace_batch(self, zenith_deg, azimuth_deg, counts, first_photon_id=0, seed=1, records=False, first_point=0):
        """One launch for the spectral points first_point .. first_point + len(counts) - 1 (slot = stream id =
        point, counts[j - first_point] photons)."""
        arr = (C.c_uint64 * len(counts))(*[int(x) for x in counts])
        total = sum(int(x) for x in counts)
        rec = torch.zeros((max(total, 1), 4), dtype=torch.int32, device=self.device) if records else None
        self._check(self.L.rt_trace_batch(self.ctx, zenith_deg, azimuth_deg, int(first_point), len(counts), arr, int(first_photon_id),
                                          int(seed), _stream(self.device), _ptr(rec)), "rt_trace_batch")
        return rec[:total] if records else None

    def trace(self, zenith_deg, azimuth_deg, n_photons, first_photon_id=0, seed=1, stream_id=0, records=False):
        if records:
            rec = torch.zeros((max(int(n_photons), 1), 4), dtype=torch.int32, device=self.device)
            self._check(self.L.rt_trace_records(self.ctx, zenith_deg, azimuth_deg, int(n_photons), int(first_photon_id),
                                                int(seed), int(stream_id), _stream(self.device), _ptr(rec)),
                        "rt_trace_records")
            return rec[:int(n_photons)]
        self._check(self.L.rt_trace(self.ctx, zenith_deg, azimuth_deg, int(n_photons), int(first_photon_id),
                                    int(seed), int(stream_id), _stream(self.device)), "rt_trace")
        return None

    def trace_range(self, zenith_deg, azimuth_deg, job_photons, range_begin, range_count, first_photon_id=0, seed=1,
                    stream_id=0, records=False):
        """include/rt.h rt_trace_range: the photons [range_begin, range_begin + range_count) of a job of job_photons."""
        rec = torch.zeros((max(int(range_count), 1), 4), dtype=torch.int32, device=self.device) if records else None
        self._check(self.L.rt_trace_range(self.ctx, zenith_deg, azimuth_deg, int(job_photons), int(first_photon_id),
                                          int(seed), int(stream_id), _stream(self.device), int(range_begin),
                                          int(range_count), _ptr(rec)), "rt_trace_range")
        return rec[:int(range_count)] if records else None

    def read_tallies(self, host=True, atm_abs=True, out=None):
        """Copy tallies out.  `out` = an earlier Tallies whose (e.g. pinned host) buffers are reused."""
        nz, ny, nx = self.shape
        if out is not None:
            a, cols = out.atm_abs, [out.sfc_dir, out.sfc_dif, out.sfc_abs, out.toa_up]
        else:
            kw = dict(dtype=torch.int64, device="cpu" if host else self.device)
            a = torch.empty((nz, ny, nx), **kw) if atm_abs else None
            cols = [torch.empty((ny, nx), **kw) for _ in range(4)]
        cnt = rt_counters()
        self._check(self.L.rt_read_tallies(self.ctx, _ptr(a), *[_ptr(t) for t in cols], C.byref(cnt)), "rt_read_tallies")
        return Tallies(a, cols[0], cols[1], cols[2], cols[3], cnt)

    def set_heating_split(self, on=True):
        """Also tally the heating by never-scattered photons (include/rt.h rt_set_heating_split)."""
        self._check(self.L.rt_set_heating_split(self.ctx, 1 if on else 0), "rt_set_heating_split")

    def read_heating_direct(self, host=True):
        nz, ny, nx = self.shape
        out = torch.empty((nz, ny, nx), dtype=torch.int64, device="cpu" if host else self.device)
        self._check(self.L.rt_read_heating_direct(self.ctx, _ptr(out)), "rt_read_heating_direct")
        return out

    def read_tallies_async(self, out, counters_buf):
        """rt_read_tallies_async into the (pinned) buffers of `out` (a Tallies; None fields are skipped) and
        into `counters_buf`, a pinned uint8 tensor of ctypes.sizeof(rt_counters) bytes.  Valid after the current
        stream has been synchronised; `counters_of(counters_buf)` then gives the rt_counters."""
        self._check(self.L.rt_read_tallies_async(self.ctx, _ptr(out.atm_abs), _ptr(out.sfc_dir), _ptr(out.sfc_dif),
                                                 _ptr(out.sfc_abs), _ptr(out.toa_up), _ptr(counters_buf),
                                                 _stream(self.device)), "rt_read_tallies_async")

    def reset_tallies(self):
        self._check(self.L.rt_reset_tallies(self.ctx, _stream(self.device)), "rt_reset_tallies")

    def read_majorant(self):
        nz, ny, nx = self.shape
        bx, by, bz = self.block
        out = torch.empty((nz // bz, ny // by, nx // bx), dtype=torch.float32)
        self._check(self.L.rt_read_majorant(self.ctx, _ptr(out)), "rt_read_majorant")
        return out

    def read_packed_optics(self):
        nz, ny, nx = self.shape
        out = torch.empty((nz, ny, nx, 4), dtype=torch.float32)
        self._check(self.L.rt_read_packed_optics(self.ctx, _ptr(out)), "rt_read_packed_optics")
        return out

    def gather_bench(self, loads_per_thread=64, footprint_voxels=0):
        ms, n = C.c_float(0), C.c_uint64(0)
        self._check(self.L.rt_gather_bench(self.ctx, loads_per_thread, int(footprint_voxels), _stream(self.device),
                                           C.byref(ms), C.byref(n)),
                    "rt_gather_bench")
        return ms.value, n.value

    def last_trace_ms(self):
        ms = C.c_float(0)
        self._check(self.L.rt_last_trace_ms(self.ctx, C.byref(ms)), "rt_last_trace_ms")
        return ms.value

    def launch_count(self):
        return int(self.L.rt_launch_count(self.ctx))

    def close(self):
        if self.ctx:
            self.L.rt_destroy(self.ctx)
            self.ctx = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def philox_words(ctr, key, device=0):
    """Philox4x32-10 words for an (n, 4) int32/uint32 counter tensor on the device."""
    ctr = ctr.contiguous()
    out = torch.empty_like(ctr)
    rc = lib().rt_philox_words(device, _ptr(ctr), key[0], key[1], _ptr(out), ctr.shape[0])
    if rc != 0:
        raise RtError("rt_philox_words failed (%d)" % rc)
    return out


def selftest_ieee(device=0):
    """include/rt.h rt_selftest_ieee: (reciprocal mismatches, square-root mismatches) over every float of the ranges."""
    a, b = C.c_uint64(0), C.c_uint64(0)
    rc = lib().rt_selftest_ieee(int(device), C.byref(a), C.byref(b))
    if rc != 0:
        raise RtError("rt_selftest_ieee failed (%d)" % rc)
    return a.value, b.value


NO_ALLOC_MAX_CELLS = 1 << 20


def majorant_no_alloc(k_ext, khat_out, block=(1, 1, 1), merge=(1, 1, 1), merge_ratio=1.25, bad_out=None):
    """include/rt.h rt_majorant_no_alloc: the majorant table of the DEVICE field k_ext [nz][ny][nx] (fp32, contiguous)
    into the caller's DEVICE tensor khat_out, with the library allocating nothing (its scratch is a fixed device array
    of NO_ALLOC_MAX_CELLS floats).  Asynchronous on the current stream; calls that overlap on the GPU race."""
    for t in (k_ext, khat_out) + ((bad_out,) if bad_out is not None else ()):
        if not (t.is_cuda and t.is_contiguous()):
            raise RtError("rt_majorant_no_alloc takes contiguous device tensors")
    if k_ext.dtype != torch.float32 or khat_out.dtype != torch.float32 or k_ext.dim() != 3:
        raise RtError("rt_majorant_no_alloc: k_ext [nz][ny][nx] and khat_out must be fp32")
    nz, ny, nx = k_ext.shape
    bx, by, bz = block
    if khat_out.numel() != (nx // bx) * (ny // by) * (nz // bz):
        raise RtError("khat_out has %d elements, expected %d" % (khat_out.numel(), (nx // bx) * (ny // by) * (nz // bz)))
    if bad_out is not None and (bad_out.dtype != torch.int32 or bad_out.numel() != 1):
        raise RtError("bad_out must be one int32")
    L = lib()
    rc = L.rt_majorant_no_alloc(_ptr(k_ext), _ptr(khat_out), _ptr(bad_out), nx, ny, nz, bx, by, bz, int(merge[0]),
                                int(merge[1]), int(merge[2]), float(merge_ratio), k_ext.device.index, _stream(k_ext.device))
    if rc != 0:
        raise RtError("rt_majorant_no_alloc failed (%d): %s" % (rc, L.rt_no_alloc_last_error().decode()))
