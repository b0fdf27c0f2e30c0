"""Parity at the FULL PLAN of BASELINE.json configs[2..4] (100M, 500M, hotspot 1B): N, Nw, support, sigma and
mesh dtype of the config, the 4-pass sort, > 4 GB mesh indexing -- in the launch configuration bench.py times
(fusion mode 2: row occupancy + split column transform fused with the w-correction).

By default every config runs with the first 5 % of its visibilities, so that the oracle (whose per-plane
FFT cost does not depend on M) finishes in about a minute per config; the full M is opt-in:

    RICK_FULL_CONFIGS=100M,500M,hotspot python -m pytest tests/test_gpu_full_configs.py -m gpu -s

(config "10M" at full size is always on: tests/test_gpu_parity.py::test_full_config_10M_image.)
The whole oracle image is computed (plane by plane, fp64) and compared through the gates of DESIGN.md
"Parity gate"; n_kept must match exactly; the sorted order is checked through properties that hold at any
size (D4' order non-decreasing, payload is a permutation: checksum) instead of a second 1e9-element sort."""
import os

import numpy as np
import pytest
import torch

from oracle import rick_oracle as O
from paper_2411_07321_b200 import binding as B
from paper_2411_07321_b200 import workloads as W

pytestmark = pytest.mark.gpu

FULL_M = [c for c in os.environ.get("RICK_FULL_CONFIGS", "").split(",") if c]
TOL = {"c64": 1e-5, "c128": 1e-10}


@pytest.mark.parametrize("name", ["100M", "500M", "hotspot"])
def test_full_plan(name):
    cfg = W.CONFIGS[name]
    if name not in FULL_M:
        cfg = W.scaled(cfg, cfg.M // 20)
    vis = W.generate(cfg, device="cuda")
    pa = W.plan_args(cfg, vis)
    im = B.Imager(dtype=cfg.dtype, M_max=vis.M, fused=2, **pa)
    assert im.fused == 2
    indirect = not im.sorted_outputs          # fp32 mesh: rick_bin gathers nothing, the gridder fetches by index
    perm = torch.empty(vis.M, dtype=torch.int32, device="cuda") if indirect else None
    im.bin(vis.u, vis.v, vis.w, vis.vis, vis.weight, perm_out=perm)   # in indirect mode perm_out is a copy, not another path
    torch.cuda.synchronize()
    n_kept = int(im.n_kept.item())
    s = im.sorted
    if not indirect:    # checksum: the sorted payload is a permutation of the kept input (sum of bit patterns, exact in int64)
        kept_sum = int(s["u"][:n_kept].view(torch.int32).to(torch.int64).sum().item())
    im.grid_(True)
    im.fft()
    im.wcorrect(True)
    torch.cuda.synchronize()
    img = im.image.cpu().numpy()
    tm = im.timings()
    rows = B.rick_plan_rows_defined(im.plan)
    hv = vis.numpy()
    del vis
    torch.cuda.empty_cache()
    oplan = O.Plan(**pa)
    okey, oi0, oj0, ok, on = O.keys(oplan, *hv)
    assert n_kept == on
    kept = okey < oplan.n_bins
    if indirect:
        # the sorted index: a permutation of the input, kept visibilities first, non-decreasing in the D4' order
        pm = perm.cpu().numpy().view(np.uint32).astype(np.int64)
        del perm
        assert np.array_equal(np.sort(pm), np.arange(pm.size))
        assert kept[pm[:n_kept]].all() and not kept[pm[n_kept:]].any()
        ssk = ((okey.astype(np.int64) * 32 + (oj0 & 31)) * 32 + (oi0 & 31))[pm[:n_kept]]
        assert np.all(np.diff(ssk) >= 0)
        del pm, ssk
    else:
        assert kept_sum == int(hv[0][kept].view(np.int32).astype(np.int64).sum())
        # the sorted payload, located again by the oracle, is non-decreasing in the D4' order
        su, sv, sw = (s[k][:n_kept].cpu().numpy() for k in ("u", "v", "w"))
        one = np.ones(n_kept, np.complex64)
        skey, si0, sj0, _, sn = O.keys(oplan, su, sv, sw, one, np.ones(n_kept, np.float32))
        assert sn == n_kept
        ssk = (skey.astype(np.int64) * 32 + (sj0 & 31)) * 32 + (si0 & 31)      # D4' order: (plane, tile, row, column)
        assert np.all(np.diff(ssk) >= 0)
        del su, sv, sw, one, skey, si0, sj0, ssk
    del okey, oi0, oj0, ok, kept
    im.close()
    del im, s
    torch.cuda.empty_cache()
    ref, n2, st = O.image(oplan, *hv, return_timing=True)
    assert n2 == n_kept
    N = cfg.N
    t = O.taper(N, cfg.support, cfg.sigma)
    inner = slice(N // 4, 3 * N // 4)
    peak = np.abs(ref[inner, inner]).max()
    assert np.isfinite(img).all()
    tt = t / t[N // 2]
    a = b = full = 0.0
    for q0 in range(0, N, 512):                       # row blocks keep the temporaries small
        tw = np.outer(tt[q0:q0 + 512], tt)
        blk = np.abs(img[q0:q0 + 512] - ref[q0:q0 + 512])
        full = max(full, float(blk.max()))
        b = max(b, float((blk * tw).max()))
        m = tw >= 1e-2
        if m.any():
            a = max(a, float(blk[m].max()))
    print(f"\nFULL PLAN {name}: M={cfg.M} n_kept={n_kept} rows defined {rows} of {cfg.Nw * N} gateA {a / peak:.3e} "
          f"gateB {b / peak:.3e} full {full / peak:.3e} "
          f"gpu_ms {({k: round(v, 3) for k, v in tm.items()})} oracle_s {({k: round(float(v), 2) for k, v in st.items()})} "
          f"threads {O.threads()}")
    assert a <= TOL[cfg.dtype] * peak and b <= TOL[cfg.dtype] * peak
