"""ctypes binding of the CPU oracle (oracle/rt_oracle.cpp).  TEST INFRASTRUCTURE.

Argument marshalling only; all arithmetic is in the C++ file.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

W0 = 1 << 32  # tally quanta per photon
FATE_ATM_ABS, FATE_SFC_ABS, FATE_TOD_EXIT, FATE_CAPPED, FATE_ROULETTE = 1, 2, 3, 4, 5
# decision kinds of the optional decision log (rt_oracle.cpp, enum DK_*)
DK_COLLIDE, DK_FACE, DK_VOXEL, DK_CLASS, DK_POLE, DK_COLUMN, DK_ALBEDO, DK_RELEVEL = 1, 2, 3, 4, 5, 6, 7, 8

COUNTER_FIELDS = ("n_photons", "n_events", "n_null", "n_rayleigh", "n_hg", "n_atm_abs",
                  "n_sfc_hits", "n_sfc_abs", "n_toa", "n_capped", "n_cell_steps", "n_relevel",
                  "n_roulette_killed", "n_roulette_kept", "capped_energy", "roulette_lost", "roulette_gained")
N_SIGNED = 3  # the last three are int64 energies


class Counters(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in COUNTER_FIELDS[:-N_SIGNED]] + [(n, C.c_int64) for n in COUNTER_FIELDS[-N_SIGNED:]]

    def asdict(self):
        return {n: int(getattr(self, n)) for n in COUNTER_FIELDS}


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        fp = C.POINTER(C.c_float)
        ip = C.POINTER(C.c_int64)
        _lib.orc_trace.restype = C.c_int
        _lib.orc_trace.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_float, C.c_float, C.c_float,
                                   C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_float, C.c_int,
                                   C.c_float, C.c_int, fp, fp, fp, fp, fp, C.c_double, C.c_double,
                                   C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32, ip, ip, ip, ip, ip, ip,
                                   C.POINTER(Counters), C.POINTER(C.c_uint32), C.c_int,
                                   C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_uint64, C.c_uint64,
                                   C.POINTER(C.c_uint8), C.POINTER(C.c_float), C.POINTER(C.c_uint32), C.c_uint32]
        _lib.orc_hardware_threads.restype = C.c_int
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


class Tallies:
    """int64 tallies in the caller-visible layout: atm_abs [nz][ny][nx], the rest [ny][nx]."""

    def __init__(self, nx, ny, nz):
        self.atm_abs = np.zeros((nz, ny, nx), dtype=np.int64)
        self.sfc_dir = np.zeros((ny, nx), dtype=np.int64)
        self.sfc_dif = np.zeros((ny, nx), dtype=np.int64)
        self.sfc_abs = np.zeros((ny, nx), dtype=np.int64)
        self.toa_up = np.zeros((ny, nx), dtype=np.int64)
        self.counters = Counters()

    def closure(self):
        """Sum of the terminal bins (must equal n_photons * W0 exactly); in weighted mode the roulette
        ledger (energy of ended photons minus energy given to survivors) is part of the balance."""
        return (int(self.atm_abs.sum()) + int(self.sfc_abs.sum()) + int(self.toa_up.sum())
                + int(self.counters.capped_energy) + int(self.counters.roulette_lost)
                - int(self.counters.roulette_gained))


def trace(grid, optics, zenith_deg, azimuth_deg, n_photons, first_photon_id=0, seed=1, stream_id=0,
          precision=64, tallies=None, records=False, n_threads=1, merge=(1, 1, 1), merge_ratio=1.25,
          weighted=False, diffuse_fraction=0.0, sobol=False, heating_split=False, margins=False, index_range=None,
          decision_log=0):
    """Run the oracle.  grid = (nx, ny, nz, dx, dy, dz, bx, by, bz); optics = dict with
    k_ext, k_ext_cloud, ssa, g ([nz][ny][nx] fp32) and sfc_albedo ([ny][nx] fp32); merge = merged-cell
    factors ((1, 1, 1) = single-level acceleration grid); weighted = the paper's absorption
    weights + Russian roulette instead of analog absorption; diffuse_fraction and
    sobol = the paper's top-of-domain source.
    margins=True also returns, as tallies.margins, the smallest relative margin of any decision each photon took
    (bookkeeping for the fp32-vs-fp64 attribution test); decision_log=K also returns tallies.decisions = (codes
    uint8 [n][K], margins float32 [n][K], counts uint32 [n]): each photon's first K decisions as kind << 4 | outcome
    (kinds: oracle.DK_*) with the margin each was taken by.  index_range=(begin, count) traces only that part of the
    n_photons-photon job (records stay indexed by the index in the job): the shards of a multi-GPU job.
    Returns (tallies, records or None, elapsed seconds of the photon loop)."""
    nx, ny, nz, dx, dy, dz, bx, by, bz = grid
    k, kp = _f32(optics["k_ext"])
    kc, kcp = _f32(optics["k_ext_cloud"])
    w, wp = _f32(optics["ssa"])
    g, gp = _f32(optics["g"])
    al, alp = _f32(optics["sfc_albedo"])
    assert k.size == nx * ny * nz and al.size == nx * ny
    t = tallies if tallies is not None else Tallies(nx, ny, nz)
    rec = np.zeros((n_photons, 4), dtype=np.uint32) if records else None
    ip = C.POINTER(C.c_int64)
    if heating_split and getattr(t, "atm_abs_direct", None) is None:
        t.atm_abs_direct = np.zeros((nz, ny, nx), dtype=np.int64)   # heating by never-scattered photons
    mg = np.full(n_photons, np.inf, dtype=np.float64) if margins else None
    rb, rn = (0, n_photons) if index_range is None else (int(index_range[0]), int(index_range[1]))
    K = int(decision_log)
    dcode = np.zeros((n_photons, K), dtype=np.uint8) if K else None
    dmarg = np.zeros((n_photons, K), dtype=np.float32) if K else None
    dcnt = np.zeros(n_photons, dtype=np.uint32) if K else None
    el = C.c_double(0.0)
    rc = lib().orc_trace(int(precision), nx, ny, nz, dx, dy, dz, bx, by, bz, int(merge[0]), int(merge[1]),
                         int(merge[2]), float(merge_ratio), int(bool(weighted)), float(diffuse_fraction), int(bool(sobol)), kp, kcp, wp, gp, alp,
                         float(zenith_deg), float(azimuth_deg), int(n_photons), int(first_photon_id),
                         int(seed), int(stream_id), t.atm_abs.ctypes.data_as(ip),
                         t.sfc_dir.ctypes.data_as(ip), t.sfc_dif.ctypes.data_as(ip),
                         t.sfc_abs.ctypes.data_as(ip), t.toa_up.ctypes.data_as(ip),
                         t.atm_abs_direct.ctypes.data_as(ip) if heating_split else None, C.byref(t.counters),
                         rec.ctypes.data_as(C.POINTER(C.c_uint32)) if records else None,
                         int(n_threads), C.byref(el),
                         mg.ctypes.data_as(C.POINTER(C.c_double)) if margins else None, rb, rn,
                         dcode.ctypes.data_as(C.POINTER(C.c_uint8)) if K else None,
                         dmarg.ctypes.data_as(C.POINTER(C.c_float)) if K else None,
                         dcnt.ctypes.data_as(C.POINTER(C.c_uint32)) if K else None, K)
    if rc != 0:
        raise ValueError("orc_trace: bad arguments (rc=%d)" % rc)
    if margins:
        t.margins = mg
    if K:
        t.decisions = (dcode, dmarg, dcnt)
    return t, rec, el.value


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def neg_log_f32(w):
    w, wp = _f32(w)
    out = np.empty_like(w)
    lib().orc_neg_log_f32(wp, out.ctypes.data_as(C.POINTER(C.c_float)), C.c_uint64(w.size))
    return out


def sincos_2pi_f32(u):
    u, up = _f32(u)
    s = np.empty_like(u)
    c = np.empty_like(u)
    fp = C.POINTER(C.c_float)
    lib().orc_sincos_2pi_f32(up, s.ctypes.data_as(fp), c.ctypes.data_as(fp), C.c_uint64(u.size))
    return s, c


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def sample_hg(g, u, precision=64, with_sine=False):
    """Polar cosine mu(u) of the Henyey-Greenstein sampler; with_sine: also sin(theta)."""
    u, up = _f64(u)
    mu = np.empty_like(u)
    sn = np.empty_like(u)
    dp = C.POINTER(C.c_double)
    lib().orc_sample_hg(int(precision), C.c_double(g), up, mu.ctypes.data_as(dp), sn.ctypes.data_as(dp),
                        C.c_uint64(u.size))
    return (mu, sn) if with_sine else mu


def sample_rayleigh(u, precision=64, with_sine=False):
    u, up = _f64(u)
    mu = np.empty_like(u)
    sn = np.empty_like(u)
    dp = C.POINTER(C.c_double)
    lib().orc_sample_rayleigh(int(precision), up, mu.ctypes.data_as(dp), sn.ctypes.data_as(dp), C.c_uint64(u.size))
    return (mu, sn) if with_sine else mu


def rotate(d, mu, u_phi, precision=64, sn=None):
    """Rotate the unit vector d by the polar angle (cosine mu, sine sn; default sqrt(1 - mu^2)) and azimuth 2 pi u_phi."""
    v = (C.c_double * 3)(*d)
    if sn is None:
        sn = float(np.sqrt(max(0.0, 1.0 - float(mu) ** 2)))
    lib().orc_rotate(int(precision), v, C.c_double(mu), C.c_double(sn), C.c_double(u_phi))
    return np.array(list(v))


def pack_optics_f32(k, kc, w, g):
    k, kp = _f32(k)
    kc, kcp = _f32(kc)
    w, wp = _f32(w)
    g, gp = _f32(g)
    out = np.empty((k.size, 4), dtype=np.float32)
    lib().orc_pack_optics_f32(kp, kcp, wp, gp, out.ctypes.data_as(C.POINTER(C.c_float)),
                              C.c_uint64(k.size))
    return out


def majorant(nx, ny, nz, bx, by, bz, k_ext, merge=(1, 1, 1), merge_ratio=1.25):
    """Majorant table [ncz][ncy][ncx]; cells of merged blocks hold -(block maximum)."""
    k, kp = _f32(k_ext)
    out = np.empty(((nz // bz), (ny // by), (nx // bx)), dtype=np.float32)
    lib().orc_majorant(nx, ny, nz, bx, by, bz, int(merge[0]), int(merge[1]), int(merge[2]),
                       C.c_float(merge_ratio), kp, out.ctypes.data_as(C.POINTER(C.c_float)))
    return out


def sobol2(k):
    """Points k of the 2-D Sobol sequence as two uint32 arrays of 32-bit fractions."""
    k = np.ascontiguousarray(k, dtype=np.uint32)
    x1 = np.empty_like(k)
    x2 = np.empty_like(k)
    up = C.POINTER(C.c_uint32)
    lib().orc_sobol2(k.ctypes.data_as(up), x1.ctypes.data_as(up), x2.ctypes.data_as(up), C.c_uint64(k.size))
    return x1, x2


def assemble_factored(k_cloud, k_abs, k_ray, cloud_ssa, cloud_g):
    """the four optical fields of a spectral point from its factors, in fp32 and in this
    order: k_ext = (k_abs[z] + k_ray[z]) + k_cloud; ssa = (k_ray[z] + cloud_ssa * k_cloud) / k_ext (0 where
    k_ext = 0); k_ext_cloud = k_cloud; g = cloud_g.  Every numpy operation below is one IEEE fp32 operation."""
    kc = np.ascontiguousarray(k_cloud, dtype=np.float32)
    ka = np.asarray(k_abs, dtype=np.float32).reshape(-1, 1, 1)
    kr = np.asarray(k_ray, dtype=np.float32).reshape(-1, 1, 1)
    k_ext = (ka + kr) + kc
    num = kr + np.float32(cloud_ssa) * kc
    with np.errstate(divide="ignore", invalid="ignore"):
        ssa = np.where(k_ext > 0, num / k_ext, np.float32(0)).astype(np.float32)
    assert k_ext.dtype == np.float32 and num.dtype == np.float32
    return {"k_ext": k_ext, "k_ext_cloud": kc, "ssa": ssa, "g": np.full(kc.shape, np.float32(cloud_g), dtype=np.float32)}


def hardware_threads():
    return int(lib().orc_hardware_threads())
