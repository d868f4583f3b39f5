"""CPU-side checks of the product's host logic: the C-ABI library loads and exports every symbol that
include/rt.h declares (no compute calls: there is no GPU here), the binding refuses to run without a GPU,
and the multi-GPU path (photon-id ranges per rank + one int64 all-reduce) is exact, on gloo, world size 2."""
import ctypes
import os
import re
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_symbols():
    txt = open(os.path.join(ROOT, "include", "rt.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(rt_[a-z_0-9]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    from paper_2208_05247_b200 import build, binding
    path = build.build()
    L = ctypes.CDLL(path)
    syms = _header_symbols()
    assert len(syms) >= 14
    for s in syms:
        assert hasattr(L, s), s
    assert sorted(binding.EXPORTS) == syms


def test_no_cpu_fallback():
    import paper_2208_05247_b200 as rt
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(rt.RtError):
        rt.Grid(32, 32, 32, 50.0, 50.0, 50.0)
    # argument checks that need no device: NULL out pointer
    assert rt.lib().rt_create_grid(None, 32, 32, 32, 50.0, 50.0, 50.0, 8, 8, 8, 0) == -1


def test_photon_ranges_partition():
    from paper_2208_05247_b200.shard import photon_range, weak_range
    for n, world in ((0, 3), (1, 4), (1000, 7), (1 << 26, 8), (12345, 1)):
        nxt = 5
        for r in range(world):
            first, count = photon_range(r, world, n, first_photon_id=5)
            assert first == nxt and count in (n // world, n // world + 1)
            nxt += count
        assert nxt == 5 + n
    seen = set()
    for step in range(3):
        for r in range(4):
            first, cnt = weak_range(r, 4, step, 10)
            assert cnt == 10 and not (seen & set(range(first, first + cnt)))
            seen |= set(range(first, first + cnt))
    assert seen == set(range(120))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_total, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle as O          # stands in for the per-GPU rt_trace_range: tests may call the oracle
    from paper_2208_05247_b200.shard import job_range, allreduce_tallies
    from rt_inputs import CONFIGS, make_optics
    cfg = CONFIGS[1]
    opt = make_optics(cfg)
    begin, count = job_range(rank, world, n_total)
    # the shard keeps the JOB's column stratification and ids (include/rt.h rt_trace_range; oracle index_range)
    t, _, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n_total, seed=3, precision=32,
                      index_range=(begin, count))
    ts = [torch.from_numpy(getattr(t, k)) for k in ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up")]
    allreduce_tallies(ts)
    if rank == 0:
        np.savez(out, **{k: v.numpy() for k, v in zip(("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up"), ts)})
    dist.destroy_process_group()


def test_two_rank_sharding_equals_the_single_call(tmp_path):
    """Two gloo ranks trace the two halves of ONE job (job-indexed ranges) and all-reduce: the merged int64
    tallies equal the single-call tallies bit for bit (so a multi-GPU run reproduces the one-GPU sample) and
    close energy exactly."""
    import oracle as O
    from rt_inputs import CONFIGS, make_optics
    n_total = 2 * 1024 * 3 + 1           # odd: the ranks get different counts; a remainder pass exists
    out = str(tmp_path / "merged.npz")
    mp.spawn(_worker, args=(2, _free_port(), n_total, out), nprocs=2, join=True)
    m = np.load(out)
    assert int(m["atm_abs"].sum()) + int(m["sfc_abs"].sum()) + int(m["toa_up"].sum()) == n_total * O.W0
    cfg = CONFIGS[1]
    one, _, _ = O.trace(cfg.grid, make_optics(cfg), cfg.zenith_deg, cfg.azimuth_deg, n_total, seed=3, precision=32)
    for k in ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up"):
        assert (m[k] == getattr(one, k)).all(), k


def test_oracle_index_ranges_tile_the_job():
    """The oracle's index_range (the shard definition both sides implement): three ragged ranges of a job with a
    remainder pass and Sobol entry points add up to the single call, record by record."""
    import oracle as O
    from rt_inputs import CONFIGS, make_optics
    cfg = CONFIGS[1]
    opt = make_optics(cfg)
    n = 3 * cfg.ncol + 333
    kw = dict(seed=9, precision=32, records=True, sobol=True, first_photon_id=(1 << 33) + 5)
    one, rec1, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, **kw)
    acc, rec = None, np.zeros_like(rec1)
    for b, cnt in ((0, 700), (700, 2 * cfg.ncol), (700 + 2 * cfg.ncol, n - 700 - 2 * cfg.ncol)):
        acc, r, _ = O.trace(cfg.grid, opt, cfg.zenith_deg, cfg.azimuth_deg, n, tallies=acc, index_range=(b, cnt), **kw)
        rec[b:b + cnt] = r[b:b + cnt]
    assert (rec == rec1).all()
    for k in ("atm_abs", "sfc_dir", "sfc_dif", "sfc_abs", "toa_up"):
        assert (getattr(acc, k) == getattr(one, k)).all()
    assert acc.counters.asdict() == one.counters.asdict()


def test_tally_to_flux_host_helper():
    """S11: quanta -> W m^-2 / W m^-3 on the host; needs no GPU.  Vacuum over a black surface from the
    oracle: every photon arrives, so the domain-mean surface flux is the top-of-domain flux; a Beer-Lambert slab:
    the column-integrated heating plus the surface flux give back the top-of-domain flux (energy in watts)."""
    import oracle as O
    import paper_2208_05247_b200 as rt
    from rt_inputs import plane_parallel
    n, F = 1 << 14, 812.5
    cfg, opt = plane_parallel(8, 8, 8, 100.0, 100.0, 50.0, 0.0, 0.0, albedo=0.0)
    t, _, _ = O.trace(cfg.grid, opt, 30.0, 0.0, n, seed=1)
    flux = rt.tally_to_flux(torch.from_numpy(t.sfc_dir), n, cfg.ncol, F)
    assert flux.shape == (8, 8) and abs(float(flux.mean()) - F) < 1e-9 * F
    cfg, opt = plane_parallel(8, 8, 8, 100.0, 100.0, 50.0, 2e-3, 0.0, albedo=0.0)
    t, _, _ = O.trace(cfg.grid, opt, 30.0, 0.0, n, seed=1)
    heat = rt.tally_to_flux(torch.from_numpy(t.atm_abs), n, cfg.ncol, F, depth=cfg.dz)      # W m^-3
    sfc = rt.tally_to_flux(torch.from_numpy(t.sfc_abs), n, cfg.ncol, F)
    assert abs(float((heat.sum(dim=0) * cfg.dz + sfc).mean()) - F) < 1e-9 * F
    assert 0.1 * F < float(sfc.mean()) < 0.9 * F
    with pytest.raises(rt.RtError):
        rt.tally_to_flux(torch.from_numpy(t.sfc_abs), 0, cfg.ncol, F)


def test_bench_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the oracle on the host cores, CPU only) prints one JSON line with the keys
    the driver reads; rank != 0 prints nothing."""
    import json
    import subprocess
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "2",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr[-500:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "photon_paths_per_s" and d["unit"] == "paths/s"
    assert d["value"] > 0 and d["higher_is_better"] is True and d["steps"] == 1 and d["n_gpus"] == 1
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert d["config"]["workload"] == "cumulus_128x128x64"
    env["RANK"] = "1"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_committed_ncu_counters_belong_to_the_kernel_as_it_stands():
    """bench.py's roofline uses profiles/trace_kernel_counters.json only for the kernel it was captured from (sha256 of
    rt_trace.cuh + rt_device.cuh).  A kernel edit without a new capture would silently fall back to the algorithmic
    model: this test makes that visible.  Also checks the fields bench.py reads."""
    import json
    sys.path.insert(0, ROOT)
    import bench
    from rt_inputs import CONFIGS
    with open(bench.COUNTERS_FILE) as f:
        entries = json.load(f)["entries"]
    sha = bench._kernel_sha16()
    assert entries and all(e["kernel_sha16"] == sha for e in entries), (sha, [e["kernel_sha16"] for e in entries])
    cfg = CONFIGS[3]
    e = bench._ncu_counters(cfg, "analog", cfg.n_photons)
    assert e is not None and e["block"] == list(cfg.block) and e["merge"] == list(cfg.merge)
    for k in ("lts_t_sectors_op_read", "dram_bytes_read", "dram_bytes_write", "inst_executed", "thread_inst_executed",
              "issue_active_pct"):
        assert e[k] > 0
    assert bench._ncu_counters(cfg, "weighted", cfg.n_photons) is not None
