"""GPU parity: the CUDA path, called through the C ABI (ctypes binding), against the CPU oracle on the
same seeded inputs.  Integer work (keys, plane indices, stable permutation, bin offsets, n_kept) is
bit-exact; images are gated as DESIGN.md "Parity gate" states (BASELINE.json north_star tolerances:
1e-5 x peak for the fp32 mesh, 1e-10 x peak for the fp64 mesh)."""
import numpy as np
import pytest
import torch

from oracle import rick_oracle as O
from paper_2411_07321_b200 import binding as B
from paper_2411_07321_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = {"c64": 1e-5, "c128": 1e-10}


def gates(img, ref, N, support, sigma):
    """-> (gate A, gate B, full-image) max abs differences relative to the inner-half peak."""
    t = O.taper(N, support, sigma)
    tw = np.outer(t, t) / t[N // 2] ** 2
    inner = slice(N // 4, 3 * N // 4)
    peak = np.abs(ref[inner, inner]).max()
    d = np.abs(img - ref)
    return d[tw >= 1e-2].max() / peak, (d * tw).max() / peak, d.max() / peak


def make(cfg_name, M, device="cuda", **plan):
    cfg = W.scaled(W.CONFIGS[cfg_name], M, **plan)
    vis = W.generate(cfg, device=device)
    pa = W.plan_args(cfg, vis)
    return cfg, vis, pa


def run_bin(im, vis):
    M = vis.M
    key = torch.empty(max(M, 1), dtype=torch.int32, device="cuda")
    perm = torch.empty(max(M, 1), dtype=torch.int32, device="cuda")
    nb = im.Nw * (im.N // 32) ** 2
    bs = torch.empty(nb + 2, dtype=torch.int64, device="cuda")
    im.bin(vis.u, vis.v, vis.w, vis.vis, vis.weight, key_out=key, perm_out=perm, bin_start_out=bs)
    torch.cuda.synchronize()
    return (key[:M].cpu().numpy().view(np.uint32), perm[:M].cpu().numpy().view(np.uint32),
            bs.cpu().numpy().view(np.uint64), int(im.n_kept.item()))


def check_bin(im, vis, pa):
    u, v, w, vv, wt = vis.numpy()
    plan = O.Plan(**pa)
    key, perm, bs, n_kept = run_bin(im, vis)
    okey, oi0, oj0, ok, on = O.keys(plan, u, v, w, vv, wt)
    assert np.array_equal(key, okey)
    assert n_kept == on
    _, _, cell_bits = B.rick_plan_sort_layout(im.plan)
    operm = O.sort_cells(oi0, oj0, ok, col_drop=10 - cell_bits)   # D4' (10 cell bits: the exact cell)
    assert np.array_equal(perm, operm)
    _, obs = O.counting_sort(okey, plan.n_bins)
    assert np.array_equal(bs, obs)
    s = im.sorted
    sel = operm[:n_kept].astype(np.int64)
    assert np.array_equal(s["u"][:n_kept].cpu().numpy(), u[sel])
    assert np.array_equal(s["v"][:n_kept].cpu().numpy(), v[sel])
    assert np.array_equal(s["w"][:n_kept].cpu().numpy(), w[sel])
    assert np.array_equal(s["vis"][:n_kept].cpu().numpy(), vv[sel])
    assert np.array_equal(s["weight"][:n_kept].cpu().numpy(), wt[sel])
    return okey, operm, n_kept


def check_bin_fused_gather(im, vis, pa):
    """rick_bin as Imager.run and bench.py call it -- no perm_out / bin_start_out, so the gather rides in the
    last one-sweep pass (k_onesweep<..., kGather>): n_kept and the five sorted arrays against the oracle's
    stable D4' order, bit for bit."""
    u, v, w, vv, wt = vis.numpy()
    plan = O.Plan(**pa)
    s = im.sorted
    for t in s.values():
        t.view(torch.uint8).fill_(0xA5)
    im.bin(vis.u, vis.v, vis.w, vis.vis, vis.weight)
    torch.cuda.synchronize()
    n_kept = int(im.n_kept.item())
    _, oi0, oj0, ok, on = O.keys(plan, u, v, w, vv, wt)
    assert n_kept == on
    _, _, cell_bits = B.rick_plan_sort_layout(im.plan)
    sel = O.sort_cells(oi0, oj0, ok, col_drop=10 - cell_bits)[:n_kept].astype(np.int64)
    assert np.array_equal(s["u"][:n_kept].cpu().numpy(), u[sel])
    assert np.array_equal(s["v"][:n_kept].cpu().numpy(), v[sel])
    assert np.array_equal(s["w"][:n_kept].cpu().numpy(), w[sel])
    assert np.array_equal(s["vis"][:n_kept].cpu().numpy().view(np.uint32), vv[sel].view(np.uint32))
    assert np.array_equal(s["weight"][:n_kept].cpu().numpy(), wt[sel])
    return n_kept


BIN_CASES = [
    ("tiny", 100_000, {}, "c128"),
    ("10M", 300_017, dict(N=512, Nw=8), "c64"),                     # ragged tail, several sort tiles
    ("10M", 1_000_003, dict(N=2048, Nw=32), "c64"),                 # 27-bit sort keys, 3 passes of 9 bits
    ("hotspot", 400_001, dict(N=1024, Nw=4), "c64"),                # support 9, 70 % in a dense core
    ("500M", 700_001, dict(N=8192, Nw=32), "c64"),                  # the 500M plan: 31-bit sort keys, 4 passes of 8 bits
]


@pytest.mark.parametrize("name,M,plan,dtype", BIN_CASES)
def test_bin_bit_exact(name, M, plan, dtype):
    cfg, vis, pa = make(name, M, dtype=dtype, **plan)
    im = B.Imager(dtype=dtype, M_max=M, alloc_mesh=False, sorted_outputs=True, **pa)
    check_bin(im, vis, pa)
    im.close()


@pytest.mark.parametrize("name,M,plan,dtype", [c for c in BIN_CASES if c[3] == "c64"])
@pytest.mark.parametrize("fused", [0, 2])
def test_bin_bit_exact_indirect(name, M, plan, dtype, fused):
    """rick_bin as bench.py and Imager.run call it on the fp32 mesh: no sorted SoA outputs, so nothing is gathered
    and the gridder fetches its records through the sorted index (indirect mode).  perm_out is a copy of that
    index: it must be the oracle's stable D4' permutation, bit for bit; keys, n_kept and bin_start as well."""
    cfg, vis, pa = make(name, M, dtype=dtype, **plan)
    im = B.Imager(dtype=dtype, M_max=M, fused=fused, alloc_mesh=False, **pa)
    assert not im.sorted_outputs
    u, v, w, vv, wt = vis.numpy()
    plan_o = O.Plan(**pa)
    key, perm, bs, n_kept = run_bin(im, vis)
    okey, oi0, oj0, ok, on = O.keys(plan_o, u, v, w, vv, wt)
    assert np.array_equal(key, okey) and n_kept == on
    _, _, cell_bits = B.rick_plan_sort_layout(im.plan)
    assert np.array_equal(perm, O.sort_cells(oi0, oj0, ok, col_drop=10 - cell_bits))
    _, obs = O.counting_sort(okey, plan_o.n_bins)
    assert np.array_equal(bs, obs)
    im.close()


@pytest.mark.parametrize("name,M,plan,dtype", BIN_CASES)
@pytest.mark.parametrize("fused", [0, 2])
def test_bin_bit_exact_fused_gather(name, M, plan, dtype, fused):
    """The variant of rick_bin the timed path runs (gather fused into the last sort pass; fusion mode 2 adds
    the row marking)."""
    cfg, vis, pa = make(name, M, dtype=dtype, **plan)
    im = B.Imager(dtype=dtype, M_max=M, fused=fused, alloc_mesh=False, sorted_outputs=True, **pa)
    n_kept = check_bin_fused_gather(im, vis, pa)
    assert 0 < n_kept <= M
    im.close()


def test_sort_many_tiles_and_hot_bin():
    """Hand-made keys: 40 sort tiles + ragged tail, one bin holding half of the data, sentinels."""
    N, Nw = 1024, 16
    pa = dict(N=N, Nw=Nw, support=7, sigma=1.0, w_min=-8.0, w_max=8.0, dl=0.25 / N)
    M = 40 * 8192 + 4321
    rng = np.random.default_rng(77)
    s = N * pa["dl"]
    u = (rng.uniform(-500, 500, M) / s).astype(np.float32)
    v = (rng.uniform(-500, 500, M) / s).astype(np.float32)
    w = rng.uniform(-8.5, 8.5, M).astype(np.float32)          # some out of range
    hot = rng.random(M) < 0.5
    u[hot] = (rng.uniform(3, 20, hot.sum()) / s).astype(np.float32)
    v[hot] = (rng.uniform(3, 20, hot.sum()) / s).astype(np.float32)
    w[hot] = 0.3
    u[::1001] = 1e9                                              # off the mesh
    t = lambda a: torch.from_numpy(a).cuda()
    vis = W.Visibilities(t(u), t(v), t(w), torch.ones(M, dtype=torch.complex64, device="cuda"),
                         torch.ones(M, dtype=torch.float32, device="cuda"))
    im = B.Imager(dtype="c64", M_max=M, sorted_outputs=True, **pa)
    okey, _, n_kept = check_bin(im, vis, pa)
    assert 0 < n_kept < M and len(np.unique(okey)) > 2000
    im.close()


@pytest.mark.parametrize("name,M,plan,dtype", [
    ("tiny", 100_000, {}, "c128"),                                   # BASELINE.json configs[0], full size
    ("tiny", 100_000, {}, "c64"),
    ("10M", 500_000, dict(N=512, Nw=8), "c64"),
    ("100M", 400_000, dict(N=512, Nw=16), "c128"),                  # wide field: the w term matters
    ("hotspot", 400_001, dict(N=1024, Nw=4), "c64"),  # support 9, sigma 1.3
])
def test_stages_and_image(name, M, plan, dtype):
    cfg, vis, pa = make(name, M, dtype=dtype, **plan)
    N, Nw = pa["N"], pa["Nw"]
    oplan = O.Plan(**pa)
    hv = vis.numpy()
    im = B.Imager(dtype=dtype, M_max=M, **pa)
    im.bin(vis.u, vis.v, vis.w, vis.vis, vis.weight)
    # --- gridding: the modulated mesh times the checkerboard is Eq. 3
    im.grid_(True)
    torch.cuda.synchronize()
    ii = np.arange(N)
    cb = np.where((ii[:, None] + ii[None, :]) & 1, -1.0, 1.0)
    g = im.grid.cpu().numpy().astype(np.complex128) * cb[None]
    og = O.grid(oplan, *hv)
    scale = np.abs(og).max()
    gerr = np.abs(g - og).max() / scale
    assert gerr <= (1e-13 if dtype == "c128" else 2e-6), gerr
    # centre-pixel invariant on the GPU mesh (needs no FFT)
    t = O.taper(N, cfg.support, cfg.sigma)
    # --- plane transform (cuFFT) against the oracle's own FFT, plane by plane
    im.fft()
    torch.cuda.synchronize()
    P = im.grid.cpu().numpy().astype(np.complex128) * cb[None]
    for k in {0, Nw // 2, Nw - 1}:
        oP = O.plane_transform(og[k])
        ref_scale = max(np.abs(oP).max(), 1e-300)
        perr = np.abs(P[k] - oP).max() / max(ref_scale, scale)
        assert perr <= (1e-12 if dtype == "c128" else 5e-6) * max(1.0, np.log2(N)), perr
    # --- image
    im.wcorrect(True)
    torch.cuda.synchronize()
    img = im.image.cpu().numpy()
    ref = O.image(oplan, *hv)
    a, b, full = gates(img, ref, N, cfg.support, cfg.sigma)
    print(f"{name}/{dtype} N={N} Nw={Nw}: grid {gerr:.2e} gateA {a:.2e} gateB {b:.2e} full {full:.2e}")
    assert a <= TOL[dtype], a
    assert b <= TOL[dtype], b
    centre = img[N // 2, N // 2] * t[N // 2] ** 2
    assert abs(centre - og.sum().real) <= (1e-11 if dtype == "c128" else 1e-5) * np.abs(og).sum()
    im.close()


def test_full_config_10M_image():
    """BASELINE.json configs[1] at full size (1e7 visibilities, 2048^2 x 32, c64) in every fusion mode:
    2 (row occupancy + own row transforms + one-sweep column kernel: what `bench.py --config 10M` times),
    1 (dense, cuFFT rows + column kernel) and 0 (2-D cuFFT + K5)."""
    cfg, vis, pa = make("10M", W.CONFIGS["10M"].M)
    ref, n_kept, _ = O.image(O.Plan(**pa), *vis.numpy(), return_timing=True)
    for fused in (2, 1, 0):
        im = B.Imager(dtype="c64", M_max=vis.M, fused=fused, **pa)
        assert im.fused == fused
        im.grid.fill_(complex(float("nan"), float("nan")))
        img = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy()
        assert int(im.n_kept.item()) == n_kept
        a, b, full = gates(img, ref, cfg.N, cfg.support, cfg.sigma)
        print(f"10M full, fusion {fused}: n_kept={n_kept} gateA {a:.2e} gateB {b:.2e} full {full:.2e}")
        assert a <= TOL["c64"] and b <= TOL["c64"], (fused, a, b)
        im.close()
        del im
        torch.cuda.empty_cache()


def test_edge_cases():
    pa = dict(N=256, Nw=8, support=7, sigma=1.0, w_min=-100.0, w_max=100.0, dl=0.2 / 256)
    oplan = O.Plan(**pa)
    im = B.Imager(dtype="c128", M_max=16, **pa)
    z32 = lambda n: torch.zeros(n, dtype=torch.float32, device="cuda")
    # empty input
    e = W.Visibilities(z32(0), z32(0), z32(0), torch.zeros(0, dtype=torch.complex64, device="cuda"), z32(0))
    img = im.run(e.u, e.v, e.w, e.vis, e.weight)
    torch.cuda.synchronize()
    assert int(im.n_kept.item()) == 0 and float(img.abs().max()) == 0.0
    # all dropped: off-mesh, out of w range, NaN / Inf in every field
    u = torch.tensor([1e9, 0, 0, float("nan"), 0, 0, 0], dtype=torch.float32, device="cuda")
    v = torch.tensor([0, -1e9, 0, 0, float("inf"), 0, 0], dtype=torch.float32, device="cuda")
    w = torch.tensor([0, 0, 101.0, 0, 0, 0, 0], dtype=torch.float32, device="cuda")
    vv = torch.ones(7, dtype=torch.complex64, device="cuda")
    vv[5] = complex(float("nan"), 0.0)
    wt = torch.ones(7, dtype=torch.float32, device="cuda")
    wt[6] = float("inf")
    img = im.run(u, v, w, vv, wt)
    torch.cuda.synchronize()
    assert int(im.n_kept.item()) == 0 and float(img.abs().max()) == 0.0
    # the hand cases of tests/golden (edges, ties, w == w_max): keys and image
    import os
    rows = [l.split("#")[0].split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "keys_hand_cases.txt"))]
    rows = [r for r in rows if r]
    u = torch.tensor([float(r[0]) for r in rows], dtype=torch.float32, device="cuda")
    v = torch.tensor([float(r[1]) for r in rows], dtype=torch.float32, device="cuda")
    w = torch.tensor([float(r[2]) for r in rows], dtype=torch.float32, device="cuda")
    n = len(rows)
    vis = W.Visibilities(u, v, w, torch.full((n,), 1 + 0.5j, dtype=torch.complex64, device="cuda"),
                         torch.ones(n, dtype=torch.float32, device="cuda"))
    key, perm, bs, n_kept = run_bin(im, vis)
    T = pa["N"] // 32
    exp = [oplan.n_bins if int(r[5]) < 0 else (int(r[5]) * T + (int(r[4]) >> 5)) * T + (int(r[3]) >> 5) for r in rows]
    assert list(key) == exp
    img = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy()
    ref = O.image(oplan, *vis.numpy())
    a, b, _ = gates(img, ref, 256, 7, 1.0)
    assert a <= 1e-10 and b <= 1e-10
    im.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_input_order_invariance(dtype):
    cfg, vis, pa = make("10M", 200_000, N=512, Nw=8, dtype=dtype)
    im = B.Imager(dtype=dtype, M_max=vis.M, **pa)
    a = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy().copy()
    g = torch.Generator(device="cpu").manual_seed(5)
    p = torch.randperm(vis.M, generator=g).cuda()
    b = im.run(vis.u[p].contiguous(), vis.v[p].contiguous(), vis.w[p].contiguous(), vis.vis[p].contiguous(),
               vis.weight[p].contiguous()).cpu().numpy()
    t = O.taper(cfg.N, cfg.support, cfg.sigma)
    tw = np.outer(t, t) / t[cfg.N // 2] ** 2
    peak = np.abs(a * tw).max()
    assert (np.abs(a - b) * tw).max() <= (1e-12 if dtype == "c128" else 1e-5) * peak
    im.close()


def test_chunked_accumulation_and_host_entry():
    """rick_grid(zero_first=0) accumulates chunks; rick_image_from_host equals the device path."""
    cfg, vis, pa = make("10M", 120_000, N=512, Nw=8, dtype="c128")
    im = B.Imager(dtype="c128", M_max=vis.M, **pa)
    whole = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy().copy()
    half = vis.M // 2
    parts = [slice(0, half), slice(half, vis.M)]
    for n, sl in enumerate(parts):
        im.bin(vis.u[sl].contiguous(), vis.v[sl].contiguous(), vis.w[sl].contiguous(), vis.vis[sl].contiguous(),
               vis.weight[sl].contiguous())
        im.grid_(zero_first=(n == 0))
    im.fft()
    im.wcorrect(True)
    torch.cuda.synchronize()
    chunked = im.image.cpu().numpy()
    t = O.taper(cfg.N, cfg.support, cfg.sigma)
    tw = np.outer(t, t) / t[cfg.N // 2] ** 2
    assert (np.abs(chunked - whole) * tw).max() <= 1e-12 * np.abs(whole * tw).max()
    host = [x.cpu().pin_memory() for x in (vis.u, vis.v, vis.w, vis.vis, vis.weight)]
    out = torch.empty((cfg.N, cfg.N), dtype=torch.float64).pin_memory()
    im.run_from_host(*host, out)
    assert (np.abs(out.numpy() - whole) * tw).max() <= 1e-12 * np.abs(whole * tw).max()
    tm = im.timings()
    assert all(tm[k] > 0 for k in ("bin", "zero", "grid", "fft", "wcorrect", "image"))
    # rick_image_from_host_chunked: ragged slices (5 and 3 of them), copies on the second stream
    for chunks in (5, 3, 2):
        out.fill_(float("nan"))
        im.run_from_host(*host, out, chunks=chunks)
        assert (np.abs(out.numpy() - whole) * tw).max() <= 1e-12 * np.abs(whole * tw).max(), chunks
    im.close()


@pytest.mark.parametrize("fused,M,plan", [
    (0, 700_001, dict(N=512, Nw=8)),
    (2, 700_001, dict(N=512, Nw=8)),
    (1, 1_000_003, dict(N=2048, Nw=32)),       # the bench plan: the image leaves in four parts
    (2, 1_000_003, dict(N=2048, Nw=32)),
    (2, 400_003, dict(N=4096, Nw=3)),          # split column transform: sweep B leaves in four column stripes
    (1, 400_003, dict(N=4096, Nw=3)),
])
def test_image_from_host_chunked_c64(fused, M, plan):
    """rick_image_from_host_chunked on the c64 mesh, plain and with row occupancy (fusion mode 2):
    the image of 7 time slices meets the oracle's gates; repeated calls reuse the staging halves; with the
    fused column kernel the image is copied out part by part while the next part is computed."""
    cfg, vis, pa = make("10M", M, dtype="c64", **plan)
    im = B.Imager(dtype="c64", M_max=M, fused=fused, **pa)
    assert im.fused == fused
    ref = O.image(O.Plan(**pa), *vis.numpy())
    host = [x.cpu().pin_memory() for x in (vis.u, vis.v, vis.w, vis.vis, vis.weight)]
    out = torch.empty((pa["N"], pa["N"]), dtype=torch.float64).pin_memory()
    for rep in range(3):
        out.fill_(float("nan"))
        im.grid.fill_(float("nan"))
        im.run_from_host(*host, out, chunks=7)
        a, b, full = gates(out.numpy(), ref, pa["N"], cfg.support, cfg.sigma)
        assert a <= TOL["c64"] and b <= TOL["c64"], (rep, a, b, full)
    im.close()


@pytest.mark.parametrize("name,M,plan", [
    ("tiny", 100_000, dict(N=256, Nw=8)),                 # radix 16 x 16
    ("10M", 300_000, dict(N=512, Nw=8)),                  # 16 x 16 x 2
    ("100M", 300_000, dict(N=1024, Nw=16)),               # 16 x 16 x 4, wide field: the w term matters
    ("10M", 1_000_003, dict(N=2048, Nw=32)),              # 16 x 16 x 8, the bench plan
])
def test_fused_column_transform(name, M, plan):
    """rick_plan_set_fusion: row cuFFT + fused column transform / w-correction equals the oracle image
    (same gates) and the unfused path; accumulate mode (zero_first = 0) adds."""
    cfg, vis, pa = make(name, M, dtype="c64", **plan)
    N = pa["N"]
    im = B.Imager(dtype="c64", M_max=M, fused=True, **pa)
    assert im.fused
    img = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy().copy()
    ref = O.image(O.Plan(**pa), *vis.numpy())
    a, b, full = gates(img, ref, N, cfg.support, cfg.sigma)
    print(f"fused {name} N={N}: gateA {a:.2e} gateB {b:.2e} full {full:.2e}")
    assert a <= TOL["c64"] and b <= TOL["c64"]
    im.grid_(True)
    im.fft()
    im.wcorrect(False)                                     # accumulate onto the image: twice the image
    torch.cuda.synchronize()
    twice = im.image.cpu().numpy()
    t = O.taper(N, cfg.support, cfg.sigma)
    tw = np.outer(t, t) / t[N // 2] ** 2
    assert (np.abs(twice - 2 * img) * tw).max() <= 2e-6 * np.abs(img * tw).max()
    im.close()
    # a c128 plan takes the split column transform (colsplit.cu); a mesh size that is not a power of two refuses
    # fusion and stays on the two-kernel path
    im2 = B.Imager(dtype="c128", M_max=16, fused=True, alloc_mesh=False, **pa)
    assert im2.fused
    im2.close()
    im2 = B.Imager(dtype="c64", M_max=16, fused=True, alloc_mesh=False, **dict(pa, N=480, dl=pa["dl"] * N / 480))
    assert not im2.fused
    im2.close()
    # so does a plan whose |w| reaches 2^28 wavelengths (the fused screen's fixed-point phase fraction)
    pa3 = dict(pa, w_min=-1.0, w_max=float(2 ** 28))
    im3 = B.Imager(dtype="c64", M_max=16, fused=True, alloc_mesh=False, **pa3)
    assert not im3.fused
    im3.close()


@pytest.mark.parametrize("name,M,plan,dtype,fused", [
    ("tiny", 100_000, {}, "c128", False),
    ("10M", 400_000, dict(N=512, Nw=8), "c64", False),
    ("10M", 400_000, dict(N=512, Nw=8), "c64", True),
    ("hotspot", 300_001, dict(N=1024, Nw=4), "c64", False),        # support 9
])
def test_kaiser_bessel_kernel(name, M, plan, dtype, fused):
    """rick_plan_set_kernel(RICK_KERNEL_KB): the paper's own gridding kernel [D6-KB, D8-KB]: mesh and
    image against the oracle, same gates as the Gaussian."""
    cfg, vis, pa = make(name, M, dtype=dtype, **plan)
    N, beta = pa["N"], 2.34 * pa["support"]
    oplan = O.Plan(kernel="kb", beta=beta, **pa)
    hv = vis.numpy()
    im = B.Imager(dtype=dtype, M_max=M, fused=fused, kernel="kb", beta=beta, **pa)
    im.bin(vis.u, vis.v, vis.w, vis.vis, vis.weight)
    im.grid_(True)
    torch.cuda.synchronize()
    ii = np.arange(N)
    cb = np.where((ii[:, None] + ii[None, :]) & 1, -1.0, 1.0)
    g = im.grid.cpu().numpy().astype(np.complex128) * cb[None]
    og = O.grid(oplan, *hv)
    gerr = np.abs(g - og).max() / np.abs(og).max()
    assert gerr <= (1e-12 if dtype == "c128" else 2e-6), gerr
    im.fft()
    im.wcorrect(True)
    torch.cuda.synchronize()
    img = im.image.cpu().numpy()
    ref = O.image(oplan, *hv)
    t = O.taper(N, cfg.support, cfg.sigma, "kb", beta)
    tw = np.outer(t, t) / t[N // 2] ** 2
    inner = slice(N // 4, 3 * N // 4)
    peak = np.abs(ref[inner, inner]).max()
    d = np.abs(img - ref)
    a, b = d[tw >= 1e-2].max() / peak, (d * tw).max() / peak
    print(f"KB {name}/{dtype} fused={fused}: grid {gerr:.2e} gateA {a:.2e} gateB {b:.2e}")
    assert a <= TOL[dtype] and b <= TOL[dtype]
    # and it is not the Gaussian image (the switch really took effect)
    gref = O.image(O.Plan(**pa), *hv)
    assert np.abs(img - gref)[inner, inner].max() > 10 * TOL[dtype] * peak
    im.close()


@pytest.mark.parametrize("name,M,plan,kernel", [
    ("10M", 400_000, dict(N=512, Nw=8), "gauss"),
    ("10M", 1_000_003, dict(N=2048, Nw=32), "gauss"),
    ("hotspot", 300_001, dict(N=1024, Nw=4), "kb"),
])
def test_fusion_mode_2_row_occupancy(name, M, plan, kernel):
    """rick_plan_set_fusion(2): only the mesh rows some footprint touches are cleared and read.  The mesh is
    pre-filled with NaN so that any read of an untouched row, or any touched row left uncleared, shows."""
    cfg, vis, pa = make(name, M, dtype="c64", **plan)
    N, beta = pa["N"], 2.34 * pa["support"]
    im = B.Imager(dtype="c64", M_max=M, fused=2, kernel=kernel, beta=beta, **pa)
    assert im.fused == 2
    im.grid.fill_(complex(float("nan"), float("nan")))
    img = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy().copy()
    oplan = O.Plan(kernel=kernel, beta=beta, **pa)
    ref = O.image(oplan, *vis.numpy())
    t = O.taper(N, cfg.support, cfg.sigma, kernel, beta)
    tw = np.outer(t, t) / t[N // 2] ** 2
    inner = slice(N // 4, 3 * N // 4)
    peak = np.abs(ref[inner, inner]).max()
    d = np.abs(img - ref)
    assert np.isfinite(img).all()
    a, b = d[tw >= 1e-2].max() / peak, (d * tw).max() / peak
    print(f"mode2 {name} N={N} {kernel}: gateA {a:.2e} gateB {b:.2e}")
    assert a <= TOL["c64"] and b <= TOL["c64"]
    # again on the same (now dirty) mesh, and in two chunks with zero_first = 0 for the second
    again = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy().copy()
    assert (np.abs(again - img) * tw).max() <= 2e-6 * np.abs(img * tw).max()
    im.grid.fill_(complex(float("nan"), float("nan")))
    half = vis.M // 2
    for n, sl in enumerate((slice(0, half), slice(half, vis.M))):
        im.bin(vis.u[sl].contiguous(), vis.v[sl].contiguous(), vis.w[sl].contiguous(), vis.vis[sl].contiguous(),
               vis.weight[sl].contiguous())
        im.grid_(zero_first=(n == 0))
    im.fft()
    im.wcorrect(True)
    torch.cuda.synchronize()
    chunked = im.image.cpu().numpy()
    assert np.isfinite(chunked).all()
    assert (np.abs(chunked - img) * tw).max() <= 2e-6 * np.abs(img * tw).max()
    im.close()


@pytest.mark.parametrize("name,M,plan,dtype,fused", [
    ("tiny", 100_000, dict(N=256, Nw=8), "c128", 1),          # 16 x 16
    ("10M", 300_000, dict(N=512, Nw=8), "c128", 2),           # 16 x 32
    ("100M", 300_000, dict(N=1024, Nw=16), "c128", 1),        # 32 x 32, wide field: the w term matters
    ("100M", 300_000, dict(N=2048, Nw=4), "c128", 2),         # 32 x 64
    ("100M", 400_000, dict(N=4096, Nw=4), "c128", 2),         # 64 x 64: the 100M plan's transform
    ("500M", 400_000, dict(N=4096, Nw=4), "c64", 1),          # 64 x 64
    ("500M", 400_000, dict(N=4096, Nw=3), "c64", 2),          # own row kernel (rowbig.cu) 64 x 64, fp32
    ("100M", 300_000, dict(N=8192, Nw=2), "c128", 2),         # own row kernel 64 x 128, fp64
    ("500M", 400_000, dict(N=8192, Nw=3), "c64", 2),          # 64 x 128: the 500M plan's transform, odd plane count
    ("hotspot", 400_001, dict(N=16384, Nw=2), "c64", 2),      # 128 x 128: the hotspot plan's transform, support 9
])
def test_split_column_transform(name, M, plan, dtype, fused):
    """rick_plan_set_fusion on plans the one-sweep column kernel cannot take (N >= 4096, or the fp64 mesh):
    cuFFT rows + sweep A (k_col_a) + sweep B fused with the w-correction (k_col_b).  Image against the oracle
    (same gates); with fusion mode 2 the mesh is pre-filled with NaN; accumulate mode adds."""
    cfg, vis, pa = make(name, M, dtype=dtype, **plan)
    N = pa["N"]
    im = B.Imager(dtype=dtype, M_max=M, fused=fused, **pa)
    assert im.fused == fused
    if fused == 2:
        im.grid.view(torch.float64 if dtype == "c128" else torch.float32).fill_(float("nan"))
    img = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy().copy()
    assert np.isfinite(img).all()
    ref = O.image(O.Plan(**pa), *vis.numpy())
    a, b, full = gates(img, ref, N, cfg.support, cfg.sigma)
    print(f"split {name}/{dtype} N={N} Nw={pa['Nw']} fusion {fused}: gateA {a:.2e} gateB {b:.2e} full {full:.2e}")
    assert a <= TOL[dtype] and b <= TOL[dtype]
    im.grid_(True)
    im.fft()
    im.wcorrect(False)                                     # accumulate onto the image: twice the image
    torch.cuda.synchronize()
    twice = im.image.cpu().numpy()
    t = O.taper(N, cfg.support, cfg.sigma)
    tw = np.outer(t, t) / t[N // 2] ** 2
    assert (np.abs(twice - 2 * img) * tw).max() <= (1e-12 if dtype == "c128" else 2e-6) * np.abs(img * tw).max()
    im.close()


@pytest.mark.parametrize("dtype,N", [("c64", 4096), ("c128", 4096)])
def test_segment_occupancy_accumulates_across_slices(dtype, N):
    """Fusion mode 2 where the long-row kernel runs keeps the occupancy per SEGMENT of a mesh row (rows.cu: 64
    segments of N / 64 cells).  A second rick_bin / rick_grid(zero_first = 0) whose visibilities fall into OTHER
    segments of rows the first one defined (left half of the uv plane, then the right half) must clear exactly those
    segments first: the mesh is pre-filled with NaN, the image of the two halves equals the image of the whole
    input, and the defined cells are the same set, sparser than the defined rows."""
    cfg, vis, pa = make("500M", 300_000, dtype=dtype, N=N, Nw=2)
    im = B.Imager(dtype=dtype, M_max=vis.M, fused=2, **pa)
    assert im.fused == 2
    real = torch.float64 if dtype == "c128" else torch.float32
    im.grid.view(real).fill_(float("nan"))
    whole = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy().copy()
    assert np.isfinite(whole).all()
    rows = B.rick_plan_rows_defined(im.plan)
    cells = B.rick_plan_cells_defined(im.plan)
    assert 0 < cells < rows * N and cells % (N // 64) == 0          # whole segments, fewer than whole rows
    ref = O.image(O.Plan(**pa), *vis.numpy())
    a, b, _ = gates(whole, ref, N, cfg.support, cfg.sigma)
    assert a <= TOL[dtype] and b <= TOL[dtype]
    im.grid.view(real).fill_(float("nan"))
    left = vis.u < 0
    seen = []
    for n, sel in enumerate((left, ~left)):
        im.bin(*(t[sel].contiguous() for t in (vis.u, vis.v, vis.w, vis.vis, vis.weight)))
        im.grid_(zero_first=(n == 0))
        torch.cuda.synchronize()
        seen.append(B.rick_plan_cells_defined(im.plan))
    assert 0 < seen[0] < seen[1] == cells
    im.fft()
    im.wcorrect(True)
    torch.cuda.synchronize()
    halves = im.image.cpu().numpy()
    assert np.isfinite(halves).all()
    t = O.taper(N, cfg.support, cfg.sigma)
    tw = np.outer(t, t) / t[N // 2] ** 2
    assert (np.abs(halves - whole) * tw).max() <= (1e-12 if dtype == "c128" else 2e-6) * np.abs(whole * tw).max()
    im.close()


@pytest.mark.parametrize("S", [3, 5, 7, 9, 11, 13, 15])
@pytest.mark.parametrize("dtype,sorted_outputs", [("c64", False), ("c64", True), ("c128", True)])
@pytest.mark.parametrize("kernel", ["gauss", "kb"])
def test_every_support(S, dtype, sorted_outputs, kernel):
    """Every footprint width rick_plan_create accepts, both mesh types, both kernels (the multi-pass record
    gridder for S >= 11 in its direct and its indirect form -- with and without the sorted outputs of rick_bin --
    and every k_grid_runs instantiation): mesh and image against the oracle.  The input
    includes visibilities on the last cells D5 keeps (i0 = h and i0 = N-1-h: the window's zero column falls
    off the row there)."""
    N, Nw, M = 256, 4, 60_000
    sigma = max(0.45, 0.16 * S)
    cfg, vis, pa = make("10M", M, dtype=dtype, N=N, Nw=Nw, support=S, sigma=sigma)
    h = (S - 1) // 2
    du = 1.0 / (N * pa["dl"])
    edge = torch.tensor([(h - N // 2) * du, (N - 1 - h - N // 2) * du], dtype=torch.float32, device="cuda")
    vis.u[:2] = edge
    vis.v[:2] = edge.flip(0)
    vis.u[2:4] = edge
    vis.v[2:4] = 0.0
    beta = 2.34 * S
    oplan = O.Plan(kernel=kernel, beta=beta, **pa)
    hv = vis.numpy()
    im = B.Imager(dtype=dtype, M_max=M, kernel=kernel, beta=beta, sorted_outputs=sorted_outputs, **pa)
    im.bin(vis.u, vis.v, vis.w, vis.vis, vis.weight)
    im.grid_(True)
    torch.cuda.synchronize()
    ii = np.arange(N)
    cb = np.where((ii[:, None] + ii[None, :]) & 1, -1.0, 1.0)
    g = im.grid.cpu().numpy().astype(np.complex128) * cb[None]
    og = O.grid(oplan, *hv)
    gerr = np.abs(g - og).max() / np.abs(og).max()
    assert gerr <= (1e-12 if dtype == "c128" else 3e-6), gerr
    im.fft()
    im.wcorrect(True)
    torch.cuda.synchronize()
    img = im.image.cpu().numpy()
    ref = O.image(oplan, *hv)
    t = O.taper(N, S, sigma, kernel, beta)
    tw = np.outer(t, t) / t[N // 2] ** 2
    inner = slice(N // 4, 3 * N // 4)
    peak = np.abs(ref[inner, inner]).max()
    d = np.abs(img - ref)
    a, b = d[tw >= 1e-2].max() / peak, (d * tw).max() / peak
    print(f"S={S} {dtype} {kernel}: grid {gerr:.2e} gateA {a:.2e} gateB {b:.2e}")
    assert a <= TOL[dtype] and b <= TOL[dtype]
    im.close()


@pytest.mark.parametrize("N,dtype", [(96, "c128"), (160, "c64"), (480, "c64")])
def test_mesh_size_not_a_power_of_two(N, dtype):
    """rick_plan_create accepts any multiple of 32.  The oracle's own FFT is radix 2, so D7 is evaluated here
    with numpy's ifft2 on the oracle's mesh (the identity tests/test_oracle_pins.py pins the oracle's transform
    with), then the oracle's own w-correction."""
    Nw, M = 4, 50_000
    cfg, vis, pa = make("10M", M, dtype=dtype, N=N, Nw=Nw)
    oplan = O.Plan(**pa)
    hv = vis.numpy()
    im = B.Imager(dtype=dtype, M_max=M, **pa)
    img = im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight).cpu().numpy()
    og = O.grid(oplan, *hv)
    ii = np.arange(N)
    cb = np.where((ii[:, None] + ii[None, :]) & 1, -1.0, 1.0)
    planes = np.stack([cb * np.fft.ifft2(cb * og[k]) * (N * N) for k in range(Nw)])
    ref = O.wcorrect(oplan, planes)
    a, b, full = gates(img, ref, N, cfg.support, cfg.sigma)
    print(f"N={N} {dtype}: gateA {a:.2e} gateB {b:.2e}")
    assert a <= TOL[dtype] and b <= TOL[dtype]
    im.close()
