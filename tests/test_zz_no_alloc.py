"""rick_bin_static (include/rick_b200.h): the allocation-free binning entry point, whose scratch is the library's
file-scope device array, against the existing path (rick_bin with a caller workspace) on the same inputs:
keys, stable permutation, bin offsets, n_kept and the sorted arrays bit for bit, and the image the rest of the
path makes from either binding within the parity tolerance of tests/test_gpu_parity.py.

Two calls in a row on different inputs: the second one finds the scratch as the first left it.
(The file name sorts last on purpose: the run is `pytest -x`.)"""
import numpy as np
import pytest
import torch

from oracle import rick_oracle as O
from paper_2411_07321_b200 import binding as B
from paper_2411_07321_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = {"c64": 1e-5, "c128": 1e-10}      # x peak of the existing path's image (BASELINE.json north_star)


def gates(img, ref, N, support, sigma):
    """the two gates of DESIGN.md "Parity gate", as in tests/test_gpu_parity.py: max abs difference where the taper
    is >= 1e-2 of its centre value (A) and taper-weighted everywhere (B), relative to the inner-half peak (two runs
    of the SAME path differ by the order of the fp32 additions on the mesh, which 1 / taper amplifies at the edge)"""
    t = O.taper(N, support, sigma)
    tw = np.outer(t, t) / t[N // 2] ** 2
    inner = slice(N // 4, 3 * N // 4)
    peak = np.abs(ref[inner, inner]).max()
    d = np.abs(img - ref)
    return d[tw >= 1e-2].max() / peak, (d * tw).max() / peak


def _inputs(cfg_name, M, dtype, **plan):
    cfg = W.scaled(W.CONFIGS[cfg_name], M, dtype=dtype, **plan)
    vis = W.generate(cfg, device="cuda")
    return cfg, vis, W.plan_args(cfg, vis)


def _outputs(im, M):
    nb = im.Nw * (im.N // 32) ** 2
    return dict(key=torch.full((max(M, 1),), -1, dtype=torch.int32, device="cuda"),
                perm=torch.full((max(M, 1),), -1, dtype=torch.int32, device="cuda"),
                bs=torch.full((nb + 2,), -1, dtype=torch.int64, device="cuda"))


def _rest_of_path(im):
    im.grid_(True)
    im.fft()
    im.wcorrect(True)
    torch.cuda.synchronize()
    return im.image.cpu().numpy().copy()


def _compare(dtype, fused, pa, calls):
    """calls: list of (u, v, w, vis, weight) device tensors, binned one after the other through both entry points."""
    M_max = max(int(c[0].numel()) for c in calls)
    ref = B.Imager(dtype=dtype, M_max=M_max, fused=fused, **pa)            # existing path: caller workspace
    new = B.Imager(dtype=dtype, M_max=1, fused=fused, **pa)                # no workspace to speak of: never passed
    assert ref.fused == new.fused == fused
    sorted_out = ref.sorted_outputs
    if sorted_out:       # the five sorted arrays are outputs of the caller in both paths
        d = "cuda"
        new_sorted = dict(u=torch.empty(M_max, dtype=torch.float32, device=d), v=torch.empty(M_max, dtype=torch.float32, device=d),
                          w=torch.empty(M_max, dtype=torch.float32, device=d), vis=torch.empty(M_max, dtype=torch.complex64, device=d),
                          weight=torch.empty(M_max, dtype=torch.float32, device=d))
    else:
        new_sorted = dict(u=None, v=None, w=None, vis=None, weight=None)
    for n_call, (u, v, w, vv, wt) in enumerate(calls):
        M = int(u.numel())
        a, b = _outputs(ref, M), _outputs(new, M)
        ref.bin(u, v, w, vv, wt, key_out=a["key"], perm_out=a["perm"], bin_start_out=a["bs"])
        img_a = _rest_of_path(ref)
        free_before = torch.cuda.mem_get_info()[0]
        B.rick_bin_static(new.plan, M, u, v, w, vv, wt, new_sorted["u"], new_sorted["v"], new_sorted["w"],
                          new_sorted["vis"], new_sorted["weight"], new.n_kept, key_out=b["key"], perm_out=b["perm"],
                          bin_start_out=b["bs"])
        torch.cuda.synchronize()
        if n_call > 0:   # every kernel is loaded by now: a call that allocated would show here
            assert torch.cuda.mem_get_info()[0] >= free_before
        img_b = _rest_of_path(new)
        n_kept = int(ref.n_kept.item())
        assert int(new.n_kept.item()) == n_kept and 0 < n_kept <= M
        for k in ("key", "perm", "bs"):
            assert torch.equal(a[k], b[k]), (n_call, k)
        if sorted_out:
            for k in ("u", "v", "w", "vis", "weight"):
                assert torch.equal(ref.sorted[k][:n_kept].view(torch.int32), new_sorted[k][:n_kept].view(torch.int32)), (n_call, k)
        assert np.isfinite(img_b).all()
        a_gate, b_gate = gates(img_b, img_a, ref.N, pa["support"], pa["sigma"])
        assert a_gate <= TOL[dtype] and b_gate <= TOL[dtype], (n_call, a_gate, b_gate)
    ref.close()
    new.close()


def _two_calls(vis, M2):
    """the whole input, then its last M2 visibilities in reverse order (other tiles, other tail, other n_kept)"""
    first = (vis.u, vis.v, vis.w, vis.vis, vis.weight)
    second = tuple(torch.flip(t[-M2:], dims=[0]).contiguous() for t in first)
    return [first, second]


def test_bin_static_matches_rick_bin_c64_indirect():
    """the configuration bench.py times: fp32 mesh, no sorted copies (the gridder fetches its records from the
    static scratch through the sorted index), fusion mode 2; M = the static maximum, then a ragged smaller call"""
    _, vis, pa = _inputs("10M", B.RICK_BIN_STATIC_MAX_M, "c64", N=1024, Nw=8)
    _compare("c64", 2, pa, _two_calls(vis, 150_001))


def test_bin_static_matches_rick_bin_c128_sorted():
    """fp64 mesh: the five sorted arrays are caller outputs, the gridder records live in the static scratch"""
    _, vis, pa = _inputs("tiny", 100_000, "c128")
    _compare("c128", 0, pa, _two_calls(vis, 33_333))


def test_bin_static_refuses_beyond_the_maximum():
    _, vis, pa = _inputs("tiny", 4096, "c64")
    im = B.Imager(dtype="c64", M_max=1, alloc_mesh=False, **pa)
    big = B.RICK_BIN_STATIC_MAX_M + 1
    f = torch.zeros(big, dtype=torch.float32, device="cuda")
    c = torch.zeros(big, dtype=torch.complex64, device="cuda")
    im.n_kept.fill_(-7)
    with pytest.raises(B.RickError, match=r"RICK_BIN_STATIC_MAX_M.*\(-6\)"):
        B.rick_bin_static(im.plan, big, f, f, f, c, f, None, None, None, None, None, im.n_kept)
    torch.cuda.synchronize()
    assert int(im.n_kept.item()) == -7          # refused before anything was enqueued
    # and the maximum itself is accepted (all-zero visibilities: every one lands in the centre cell of plane w = 0, or is dropped)
    B.rick_bin_static(im.plan, big - 1, f, f, f, c, f, None, None, None, None, None, im.n_kept)
    torch.cuda.synchronize()
    assert 0 <= int(im.n_kept.item()) <= big - 1
    # M = 0 binds an empty set
    B.rick_bin_static(im.plan, 0, f, f, f, c, f, None, None, None, None, None, im.n_kept)
    torch.cuda.synchronize()
    assert int(im.n_kept.item()) == 0
    im.close()
