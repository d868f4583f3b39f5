"""rt_majorant_no_alloc (include/rt.h): the majorant table for callers that cannot call cudaMalloc.  Its scratch (the
per-cell minima of the merge criterion) lives in a fixed file-scope device array, so every call shares it and it keeps
the last call's contents.  Checked here against the existing path (rt_set_optics + rt_read_majorant on a context) bit
for bit -- the bar the other majorant tests use (tests/test_gpu_parity.py) -- on calls in a row whose cell grids differ
in size, so that a table built from stale scratch would show.  This file is collected last on purpose."""
import numpy as np
import pytest
import torch

from rt_inputs import CONFIGS, make_optics

pytestmark = pytest.mark.gpu
NAMES = ("k_ext", "k_ext_cloud", "ssa", "g", "sfc_albedo")


def _rt():
    import paper_2208_05247_b200 as rt
    return rt


def _existing_path(rt, cfg, opt, block, merge):
    g = rt.Grid(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, *block, device=0, merge=merge, merge_ratio=cfg.merge_ratio)
    g.set_optics(*[opt[k] for k in NAMES])
    kh = g.read_majorant().numpy().copy()
    g.close()
    return kh


def test_majorant_no_alloc_equals_the_context_path_on_calls_in_a_row():
    rt = _rt()
    cases = [(CONFIGS[2], (1, 1, 1), (8, 8, 8)),      # 2^20 cells: exactly RT_NO_ALLOC_MAX_CELLS, both levels in use
             (CONFIGS[1], (2, 2, 2), (4, 4, 4)),      # 4096 cells right after: stale minima lie beyond and around them
             (CONFIGS[2], (4, 4, 4), (1, 1, 1)),      # no merging: the scratch is written and not read
             (CONFIGS[2], (1, 1, 1), (8, 8, 8))]      # the first case again, on what the others left behind
    opts = {id(c): make_optics(c) for c in (CONFIGS[1], CONFIGS[2])}
    want = [_existing_path(rt, cfg, opts[id(cfg)], blk, mrg) for cfg, blk, mrg in cases]
    assert (want[0] < 0).any() and (want[0] > 0).any()          # merged and single cells both occur
    dev = torch.device("cuda", 0)
    fields = {id(c): torch.from_numpy(opts[id(c)]["k_ext"]).to(dev) for c in (CONFIGS[1], CONFIGS[2])}
    outs = [torch.empty(w.size, dtype=torch.float32, device=dev) for w in want]     # the caller's buffers, made up front
    bad = torch.ones(1, dtype=torch.int32, device=dev)
    for (cfg, blk, mrg), out in zip(cases, outs):               # back to back on one stream, nothing read in between
        rt.majorant_no_alloc(fields[id(cfg)], out, block=blk, merge=mrg, merge_ratio=cfg.merge_ratio, bad_out=bad)
    torch.cuda.synchronize()
    assert int(bad.item()) == 0
    for k, (out, w) in enumerate(zip(outs, want)):
        assert np.array_equal(out.cpu().numpy().view(np.uint32), w.reshape(-1).view(np.uint32)), k


def test_majorant_no_alloc_limits_and_flags():
    rt = _rt()
    dev = torch.device("cuda", 0)
    k = torch.rand((128, 128, 128), dtype=torch.float32, device=dev)
    out = torch.empty(128 ** 3, dtype=torch.float32, device=dev)
    with pytest.raises(rt.RtError, match="RT_NO_ALLOC_MAX_CELLS"):          # 2^21 voxel-sized cells: beyond the array
        rt.majorant_no_alloc(k, out, block=(1, 1, 1), merge=(8, 8, 8))
    with pytest.raises(rt.RtError, match="merge factors"):
        rt.majorant_no_alloc(k, out[: 64 ** 3], block=(2, 2, 2), merge=(3, 1, 1))
    # 2^18 cells of 2^3 voxels fit; a bad value is flagged on the device, a second call clears the flag
    bad = torch.zeros(1, dtype=torch.int32, device=dev)
    kb = k.clone()
    kb[5, 6, 7] = -1.0
    rt.majorant_no_alloc(kb, out[: 64 ** 3], block=(2, 2, 2), merge=(8, 8, 8), bad_out=bad)
    assert int(bad.item()) == 1
    rt.majorant_no_alloc(k, out[: 64 ** 3], block=(2, 2, 2), merge=(8, 8, 8), bad_out=bad)
    assert int(bad.item()) == 0
    # against plain torch on this field (uniform random: no block merges at ratio 1.25, every cell keeps its own maximum)
    ref = k.reshape(64, 2, 64, 2, 64, 2).amax(dim=(1, 3, 5)).reshape(-1)
    assert torch.equal(out[: 64 ** 3], ref)
