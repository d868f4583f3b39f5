"""The seeded input generators (rt_inputs) produce what BASELINE.json's configs describe:
shapes, magnitudes, cloud cover, the spectral points and the photon split.  No method arithmetic here."""
import numpy as np

from rt_inputs import CONFIGS, make_optics, spectral_points, split_photons


def test_config_shapes_and_ranges():
    for key, (grid, ncol_photons) in {1: ((32, 32, 32), 256), 2: ((128, 128, 64), 256)}.items():
        cfg = CONFIGS[key]
        assert (cfg.nx, cfg.ny, cfg.nz) == grid and cfg.n_photons == ncol_photons * cfg.ncol
        opt = make_optics(cfg)
        for k in ("k_ext", "k_ext_cloud", "ssa", "g"):
            assert opt[k].shape == (cfg.nz, cfg.ny, cfg.nx) and opt[k].dtype == np.float32
        assert opt["sfc_albedo"].shape == (cfg.ny, cfg.nx)
        assert (opt["k_ext"] > 0).all() and (opt["k_ext_cloud"] <= opt["k_ext"]).all()
        assert (opt["ssa"] >= 0).all() and (opt["ssa"] <= 1).all() and (np.abs(opt["g"]) < 1).all()
    # config 1: the 8^3 cube of extinction 0.02 at voxels 12..19, uniform gas 2e-5 + 1e-5 (BASELINE.json configs[0])
    opt = make_optics(CONFIGS[1])
    cube = opt["k_ext_cloud"] > 0
    assert cube.sum() == 512 and cube[12:20, 12:20, 12:20].all()
    assert np.allclose(opt["k_ext"][~cube], 3e-5) and np.allclose(opt["k_ext_cloud"][cube], 0.02)
    # config 2: gas falls off with an 8 km scale height; clouds between 600 m and the top minus two levels;
    # median cloud extinction about 0.05 1/m; same field on every call (seeded)
    cfg = CONFIGS[2]
    opt = make_optics(cfg)
    gas = opt["k_ext"] - opt["k_ext_cloud"]
    assert abs(gas[0, 0, 0] / gas[-1, 0, 0] - np.exp((cfg.nz - 1) * cfg.dz / 8000.0)) < 1e-3
    cloudy = opt["k_ext_cloud"] > 0
    levels = np.nonzero(cloudy.any(axis=(1, 2)))[0]
    assert levels.min() * cfg.dz >= 575.0 and levels.max() <= cfg.nz - 2
    assert 0.03 < np.median(opt["k_ext_cloud"][cloudy]) < 0.08
    cover = cloudy.any(axis=0).mean()
    assert 0.1 < cover < 0.45, cover                       # ~26 % expected; 40 blobs: large sampling spread
    assert np.array_equal(make_optics(cfg)["k_ext"], opt["k_ext"])


def test_spectral_points_and_photon_split():
    pts = spectral_points(112)
    lam = np.array([p["lambda_um"] for p in pts])
    assert len(pts) == 112 and abs(lam[0] - 0.2) < 1e-12 and abs(lam[-1] - 4.0) < 1e-9
    assert np.all(np.diff(np.log(lam)) > 0) and np.allclose(np.diff(np.log(lam)), np.log(20.0) / 111)
    kabs = np.array([p["k_abs0"] for p in pts])
    assert kabs.min() >= 1e-7 and kabs.max() <= 1e-3
    kray = np.array([p["k_ray0"] for p in pts])
    assert np.allclose(kray * lam ** 4, kray[0] * lam[0] ** 4)          # lambda^-4
    assert abs(pts[0]["cloud_ssa"] - 0.9999) < 1e-12 and abs(pts[-1]["cloud_ssa"] - 0.9) < 1e-12
    assert abs(pts[0]["cloud_g"] - 0.86) < 1e-12 and abs(pts[-1]["cloud_g"] - 0.80) < 1e-12
    w = np.array([p["weight"] for p in pts])
    assert abs(w.sum() - 1) < 1e-12 and (w > 0).all()
    n = 1 << 26
    counts = split_photons(n, w)
    assert sum(counts) == n and all(abs(c - n * x) < 1 for c, x in zip(counts, w))
    assert split_photons(7, [1, 1, 1]) == [3, 2, 2] and split_photons(0, [1, 2]) == [0, 0]


def test_factored_point_is_the_same_point():
    """The factored form of a spectral point (cloud field + gas profiles, assembled in fp32 by DESIGN.md §3.4b)
    describes the same optics as the full fields of make_optics (assembled in fp64, rounded once): equal to
    fp32 rounding."""
    import oracle as O
    from rt_inputs import factored_point
    cfg = CONFIGS[2]
    p = spectral_points(112)[60]
    full = make_optics(cfg, p)
    f = factored_point(cfg, p)
    asm = O.assemble_factored(f["k_cloud"], f["k_abs"], f["k_ray"], f["cloud_ssa"], f["cloud_g"])
    assert np.array_equal(asm["k_ext_cloud"], full["k_ext_cloud"]) and np.array_equal(asm["g"], full["g"])
    for k in ("k_ext", "ssa"):
        rel = np.abs(asm[k].astype(np.float64) - full[k]) / np.maximum(np.abs(full[k]), 1e-30)
        assert rel.max() < 4e-7, (k, rel.max())
    assert np.array_equal(f["sfc_albedo"], full["sfc_albedo"])
