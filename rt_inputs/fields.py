"""Synthetic optical-property fields (numpy only).  See DESIGN.md §4 for the recipe."""
from dataclasses import dataclass, replace

import numpy as np

FIELD_SEED = 2208
SCALE_HEIGHT = 8000.0  # m


@dataclass(frozen=True)
class Config:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    zenith_deg: float
    azimuth_deg: float
    n_photons: int
    sfc_albedo: float
    n_blobs: int = 0
    k_abs0: float = 1.5e-5     # gas absorption at the surface, 1/m
    k_ray0: float = 1.2e-5     # Rayleigh scattering at the surface, 1/m
    cloud_ssa: float = 0.9999
    cloud_g: float = 0.86
    seed: int = 1              # Philox trace seed
    block: tuple = (8, 8, 8)   # acceleration-grid block, voxels (Q1: the paper gives no size; on the
                               # LES-scale fields voxel-sized cells merged 8^3 in clear air are the fastest, profiles/)
    merge: tuple = (1, 1, 1)   # merged acceleration cells: blocks of this many cells with
    merge_ratio: float = 1.25  # max k_ext <= merge_ratio * min k_ext are traversed as one cell

    @property
    def grid(self):
        return (self.nx, self.ny, self.nz, self.dx, self.dy, self.dz) + tuple(self.block)

    @property
    def accel(self):
        """Keyword arguments of the merged-cell setting, for rt.Grid(...) and oracle.trace(...)."""
        return {"merge": tuple(self.merge), "merge_ratio": self.merge_ratio}

    @property
    def ncol(self):
        return self.nx * self.ny

    @property
    def nvox(self):
        return self.nx * self.ny * self.nz


# BASELINE.json configs[0..4] (config 4 = config 3's field traced at 112 spectral points).
CONFIGS = {
    1: Config("tiny_box_32", 32, 32, 32, 50.0, 50.0, 50.0, 30.0, 0.0, 1 << 18, 0.2,
              k_abs0=2e-5, k_ray0=1e-5, cloud_ssa=0.999, cloud_g=0.85),
    2: Config("cumulus_128x128x64", 128, 128, 64, 50.0, 50.0, 25.0, 45.0, 0.0, 1 << 22, 0.2, n_blobs=40,
              block=(4, 4, 4)),
    3: Config("cumulus_512x512x128", 512, 512, 128, 50.0, 50.0, 25.0, 60.0, 120.0, 1 << 26, 0.2,
              n_blobs=600, block=(1, 1, 1), merge=(8, 8, 8)),
    4: Config("spectral_512x512x128", 512, 512, 128, 50.0, 50.0, 25.0, 60.0, 120.0, 1 << 26, 0.2,
              n_blobs=600, block=(1, 1, 1), merge=(8, 8, 8)),
    5: Config("convergence_1024x1024x192", 1024, 1024, 192, 25.0, 25.0, 20.0, 50.0, 0.0, 1 << 28, 0.15,
              n_blobs=2400, block=(1, 1, 1), merge=(8, 8, 8)),
}


def _cloud_k(cfg: Config) -> np.ndarray:
    """Cloud extinction [nz][ny][nx] (float64): flat-based half-ellipsoid blobs with lognormal
    liquid water, k = 3 LWC rho_air / (2 rho_w r_e)."""
    nx, ny, nz = cfg.nx, cfg.ny, cfg.nz
    kc = np.zeros((nz, ny, nx), dtype=np.float64)
    if cfg.n_blobs == 0:
        return kc
    rng = np.random.Generator(np.random.Philox(key=FIELD_SEED))
    Lx, Ly = nx * cfg.dx, ny * cfg.dy
    r0 = np.sqrt(0.3 * Lx * Ly / (np.pi * cfg.n_blobs))
    top_max = (nz - 2) * cfg.dz
    mask = np.zeros((nz, ny, nx), dtype=bool)
    zc = (np.arange(nz) + 0.5) * cfg.dz
    for _ in range(cfg.n_blobs):
        xc, yc = rng.uniform(0, Lx), rng.uniform(0, Ly)
        base = rng.uniform(600.0, 800.0)
        depth = rng.uniform(200.0, 1000.0)
        a, b = rng.uniform(0.6, 1.4) * r0, rng.uniform(0.6, 1.4) * r0
        depth = min(depth, top_max - base)
        if depth <= 0:
            continue
        # bounding box in voxel indices (periodic in x, y)
        i0, i1 = int(np.floor((xc - a) / cfg.dx)), int(np.ceil((xc + a) / cfg.dx))
        j0, j1 = int(np.floor((yc - b) / cfg.dy)), int(np.ceil((yc + b) / cfg.dy))
        k0, k1 = max(0, int(np.floor(base / cfg.dz))), min(nz, int(np.ceil((base + depth) / cfg.dz)) + 1)
        ii = np.arange(i0, i1 + 1)
        jj = np.arange(j0, j1 + 1)
        ex = (((ii + 0.5) * cfg.dx - xc) / a) ** 2
        ey = (((jj + 0.5) * cfg.dy - yc) / b) ** 2
        ez = ((zc[k0:k1] - base) / depth) ** 2
        inside = (ez[:, None, None] + ey[None, :, None] + ex[None, None, :] <= 1.0) & \
                 (zc[k0:k1] >= base)[:, None, None]
        sub = mask[k0:k1][:, jj % ny][:, :, ii % nx]
        sub |= inside
        # fancy indexing copies: write back
        mask[np.ix_(np.arange(k0, k1), jj % ny, ii % nx)] = sub
    ncloudy = int(mask.sum())
    noise = np.random.Generator(np.random.Philox(key=FIELD_SEED + 1)).standard_normal(ncloudy)
    lwc = 0.3e-3 * np.exp(0.6 * noise)                      # kg/kg, median 0.3 g/kg
    zz = np.broadcast_to(zc[:, None, None], mask.shape)[mask]
    rho_air = 1.2 * np.exp(-zz / SCALE_HEIGHT)
    kc[mask] = 3.0 * lwc * rho_air / (2.0 * 1000.0 * 10e-6)
    return kc


def _assemble(cfg: Config, kc: np.ndarray, k_abs0, k_ray0, cloud_ssa, cloud_g):
    zc = (np.arange(cfg.nz) + 0.5) * cfg.dz
    if cfg.name.startswith("tiny_box"):
        prof = np.ones(cfg.nz)
    else:
        prof = np.exp(-zc / SCALE_HEIGHT)
    k_abs = (k_abs0 * prof)[:, None, None]
    k_ray = (k_ray0 * prof)[:, None, None]
    k_ext = k_abs + k_ray + kc
    ssa = (k_ray + cloud_ssa * kc) / k_ext
    return {
        "k_ext": k_ext.astype(np.float32),
        "k_ext_cloud": kc.astype(np.float32),
        "ssa": ssa.astype(np.float32),
        "g": np.full(kc.shape, cloud_g, dtype=np.float32),
        "sfc_albedo": np.full((cfg.ny, cfg.nx), cfg.sfc_albedo, dtype=np.float32),
    }


_cloud_cache = {}


def make_optics(cfg: Config, spectral=None):
    """Library inputs for a configuration: dict of k_ext, k_ext_cloud, ssa, g ([nz][ny][nx] fp32)
    and sfc_albedo ([ny][nx] fp32).  `spectral` = one entry of spectral_points() or None."""
    key = (cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, cfg.n_blobs, cfg.name.startswith("tiny_box"))
    if key not in _cloud_cache:
        _cloud_cache.clear()
        if cfg.name.startswith("tiny_box"):
            kc = np.zeros((cfg.nz, cfg.ny, cfg.nx))
            kc[12:20, 12:20, 12:20] = 0.02
        else:
            kc = _cloud_k(cfg)
        _cloud_cache[key] = kc
    kc = _cloud_cache[key]
    if spectral is None:
        return _assemble(cfg, kc, cfg.k_abs0, cfg.k_ray0, cfg.cloud_ssa, cfg.cloud_g)
    return _assemble(cfg, kc, spectral["k_abs0"], spectral["k_ray0"], spectral["cloud_ssa"],
                     spectral["cloud_g"])


def factored_point(cfg: Config, spectral=None):
    """The same spectral point as make_optics(cfg, spectral), as FACTORS: cloud extinction field (fp32, shared by
    all points) and per-level gas absorption / Rayleigh profiles (fp32), cloud single-scattering albedo and g."""
    key = (cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, cfg.n_blobs, cfg.name.startswith("tiny_box"))
    if key not in _cloud_cache:
        make_optics(cfg)
    p = spectral or {"k_abs0": cfg.k_abs0, "k_ray0": cfg.k_ray0, "cloud_ssa": cfg.cloud_ssa, "cloud_g": cfg.cloud_g}
    zc = (np.arange(cfg.nz) + 0.5) * cfg.dz
    prof = np.ones(cfg.nz) if cfg.name.startswith("tiny_box") else np.exp(-zc / SCALE_HEIGHT)
    return {"k_cloud": _cloud_cache[key].astype(np.float32), "k_abs": (p["k_abs0"] * prof).astype(np.float32),
            "k_ray": (p["k_ray0"] * prof).astype(np.float32), "cloud_ssa": float(np.float32(p["cloud_ssa"])),
            "cloud_g": float(np.float32(p["cloud_g"])),
            "sfc_albedo": np.full((cfg.ny, cfg.nx), cfg.sfc_albedo, dtype=np.float32)}


def spectral_points(n=112):
    """Config 4: n spectral points, 0.2-4 um log-spaced; gas absorption log-uniform 1e-7..1e-3 1/m,
    Rayleigh ~ lambda^-4, cloud ssa 0.9999 -> 0.9 and g 0.86 -> 0.80; weight = Planck(5772 K) * dlambda
    * (0.5 + u')."""
    rng = np.random.Generator(np.random.Philox(key=FIELD_SEED + 2))
    j = np.arange(n)
    lam = 0.2 * 20.0 ** (j / (n - 1))                       # um
    edges = 0.2 * 20.0 ** ((np.arange(n + 1) - 0.5) / (n - 1))
    dlam = np.diff(edges)
    u = rng.uniform(size=n)
    u2 = rng.uniform(size=n)
    h, c, kB, T = 6.62607015e-34, 2.99792458e8, 1.380649e-23, 5772.0
    lm = lam * 1e-6
    planck = 2 * h * c ** 2 / lm ** 5 / np.expm1(h * c / (lm * kB * T))
    w = planck * dlam * (0.5 + u2)
    w = w / w.sum()
    pts = []
    for i in range(n):
        f = i / (n - 1)
        pts.append({"index": i, "lambda_um": float(lam[i]), "k_ray0": float(1.2e-5 * (lam[i] / 0.55) ** -4),
                    "k_abs0": float(10.0 ** (-7.0 + 4.0 * u[i])),
                    "cloud_ssa": float(0.9999 + f * (0.9 - 0.9999)), "cloud_g": float(0.86 + f * (0.80 - 0.86)),
                    "weight": float(w[i])})
    return pts


def split_photons(n_total, weights):
    """Largest-remainder split of n_total photons in proportion to weights."""
    w = np.asarray(weights, dtype=np.float64)
    exact = n_total * w / w.sum()
    base = np.floor(exact).astype(np.int64)
    rem = int(n_total - base.sum())
    order = np.argsort(-(exact - base), kind="stable")
    base[order[:rem]] += 1
    return [int(x) for x in base]


def plane_parallel(nx, ny, nz, dx, dy, dz, k_ext, ssa, g=0.0, cloud_frac=0.0, albedo=0.0,
                   block=(8, 8, 8), **kw):
    """Homogeneous (or per-level) slab for the analytic pins: k_ext, ssa scalars or [nz] profiles."""
    k = np.broadcast_to(np.asarray(k_ext, dtype=np.float64).reshape(-1, 1, 1), (nz, ny, nx))
    w = np.broadcast_to(np.asarray(ssa, dtype=np.float64).reshape(-1, 1, 1), (nz, ny, nx))
    cfg = Config("plane_parallel", nx, ny, nz, dx, dy, dz, kw.get("zenith_deg", 0.0),
                 kw.get("azimuth_deg", 0.0), kw.get("n_photons", 0), albedo, block=tuple(block))
    opt = {
        "k_ext": np.ascontiguousarray(k, dtype=np.float32),
        "k_ext_cloud": np.ascontiguousarray(k * cloud_frac, dtype=np.float32),
        "ssa": np.ascontiguousarray(w, dtype=np.float32),
        "g": np.full((nz, ny, nx), g, dtype=np.float32),
        "sfc_albedo": np.full((ny, nx), albedo, dtype=np.float32),
    }
    return cfg, opt


def with_photons(cfg: Config, n):
    return replace(cfg, n_photons=int(n))


def make_optics_torch(cfg: Config, spectral=None, device="cuda"):
    """make_optics() assembled on a torch device (same IEEE fp64 operations in the same order, then one
    rounding to fp32), for sweeps that re-set the optics many times (config 4).  The cloud field comes from
    the numpy generator and is cached on the device."""
    import torch
    make_optics(cfg) if spectral is None else None        # fills the host cloud cache if needed
    key = (cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, cfg.n_blobs, cfg.name.startswith("tiny_box"))
    if key not in _cloud_cache:
        make_optics(cfg)
    dkey = key + (str(device),)
    if dkey not in _cloud_cache_dev:
        _cloud_cache_dev.clear()
        _cloud_cache_dev[dkey] = torch.from_numpy(_cloud_cache[key]).to(device)
    kc = _cloud_cache_dev[dkey]
    p = spectral or {"k_abs0": cfg.k_abs0, "k_ray0": cfg.k_ray0, "cloud_ssa": cfg.cloud_ssa, "cloud_g": cfg.cloud_g}
    zc = (np.arange(cfg.nz) + 0.5) * cfg.dz
    prof = np.ones(cfg.nz) if cfg.name.startswith("tiny_box") else np.exp(-zc / SCALE_HEIGHT)
    k_abs = torch.from_numpy(p["k_abs0"] * prof).to(device)[:, None, None]
    k_ray = torch.from_numpy(p["k_ray0"] * prof).to(device)[:, None, None]
    k_ext = k_abs + k_ray + kc
    ssa = (k_ray + p["cloud_ssa"] * kc) / k_ext
    return {
        "k_ext": k_ext.float(),
        "k_ext_cloud": kc.float(),
        "ssa": ssa.float(),
        "g": torch.full(kc.shape, p["cloud_g"], dtype=torch.float32, device=device),
        "sfc_albedo": torch.full((cfg.ny, cfg.nx), cfg.sfc_albedo, dtype=torch.float32, device=device),
    }


_cloud_cache_dev = {}
