"""CPU pins for the oracle (oracle/rick_oracle.cpp): every stage is checked against something other
than itself -- hand-computed cases, closed forms, invariants, numpy library routines and a brute-force
direct DFT (SURVEY.md section 8(c) "Pins"; readings D1-D9 restated in DESIGN.md)."""
import math
import os

import numpy as np
import pytest
from scipy import integrate

from oracle import rick_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rand_vis(rng, M, N, fov, w_lo, w_hi, margin=6.0):
    """Random uvw well inside the mesh (so nothing is dropped unless the test wants it)."""
    du = 1.0 / fov
    lim = (N / 2 - margin) * du
    u = rng.uniform(-lim, lim, M).astype(np.float32)
    v = rng.uniform(-lim, lim, M).astype(np.float32)
    w = rng.uniform(w_lo, w_hi, M).astype(np.float32)
    return u, v, w


def _snap_w(plan, w):
    """Move each w to the centre of its plane (then nearest-plane stacking is exact)."""
    dw = (plan.w_max - plan.w_min) / plan.Nw
    k = np.clip(np.floor((w.astype(np.float64) - plan.w_min) / dw), 0, plan.Nw - 1)
    return (plan.w_min + (k + 0.5) * dw).astype(np.float32)


def _point_vis(u, v, w, l0, m0, amp=1.0):
    """Eq. 1 for one point source, fp64 phases on the fp32 coordinates."""
    n0m1 = math.sqrt(1.0 - l0 * l0 - m0 * m0) - 1.0
    ph = -2.0 * np.pi * (u.astype(np.float64) * l0 + v.astype(np.float64) * m0 + w.astype(np.float64) * n0m1)
    return (amp * np.exp(1j * ph)).astype(np.complex64)


# ------------------------------------------------------------------------------------------------
# keys, planes, drop rule, sort (exact)
# ------------------------------------------------------------------------------------------------

def test_keys_hand_cases_from_golden_file():
    """tests/golden/keys_hand_cases.txt: cases worked out by hand from D2-D5."""
    plan = O.Plan(N=256, Nw=8, support=7, sigma=1.0, w_min=-100.0, w_max=100.0, dl=0.2 / 256)
    rows = []
    with open(os.path.join(GOLDEN, "keys_hand_cases.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    assert len(rows) >= 12
    u = np.array([float(r[0]) for r in rows], np.float32)
    v = np.array([float(r[1]) for r in rows], np.float32)
    w = np.array([float(r[2]) for r in rows], np.float32)
    vis = np.ones(len(rows), np.complex64)
    wt = np.ones(len(rows), np.float32)
    key, i0, j0, k, n_kept = O.keys(plan, u, v, w, vis, wt)
    T = plan.T
    for n, r in enumerate(rows):
        ei0, ej0, ek = int(r[3]), int(r[4]), int(r[5])
        assert (i0[n], j0[n], k[n]) == (ei0, ej0, ek), (n, r, i0[n], j0[n], k[n])
        exp_key = plan.n_bins if ek < 0 else (ek * T + (ej0 >> 5)) * T + (ei0 >> 5)
        assert key[n] == exp_key
    assert n_kept == sum(1 for r in rows if int(r[5]) >= 0)


def test_plane_boundaries_and_nonfinite():
    plan = O.Plan(N=256, Nw=8, support=7, sigma=1.0, w_min=-100.0, w_max=100.0, dl=0.2 / 256)
    b = np.float32(-75.0)   # boundary between planes 0 and 1 (dw = 25)
    w = np.array([b, np.nextafter(b, np.float32(-np.inf)), np.nextafter(np.float32(100.0), np.float32(np.inf)),
                  np.nextafter(np.float32(-100.0), np.float32(-np.inf))], np.float32)
    z = np.zeros_like(w)
    _, _, _, k, _ = O.keys(plan, z, z, w, np.ones(4, np.complex64), np.ones(4, np.float32))
    assert list(k) == [1, 0, -1, -1]
    # non-finite in any of the six numbers drops the visibility
    one = np.ones(6, np.float32)
    u, v, w6, wt = one * 0, one * 0, one * 0, one.copy()
    vis = np.ones(6, np.complex64)
    u[0] = np.nan; v[1] = np.inf; w6[2] = -np.inf; wt[3] = np.nan
    vis[4] = complex(np.nan, 0.0); vis[5] = complex(0.0, np.inf)
    key, *_ , n_kept = O.keys(plan, u, v, w6, vis, wt)
    assert n_kept == 0 and np.all(key == plan.n_bins)


def test_key_formula_against_numpy_restatement():
    """Bulk check of D2-D4 against the same rules typed with numpy's correctly-rounded double ops
    (numpy has no fma: x is formed in longdouble, which is exact here, then rounded once)."""
    rng = np.random.default_rng(5)
    plan = O.Plan(N=512, Nw=16, support=9, sigma=1.3, w_min=-321.5, w_max=777.25, dl=0.37 / 512)
    M = 20000
    du = 1.0 / (plan.N * plan.dl)
    u = rng.uniform(-270 * du, 270 * du, M).astype(np.float32)
    v = rng.uniform(-270 * du, 270 * du, M).astype(np.float32)
    w = rng.uniform(-400, 850, M).astype(np.float32)
    key, i0, j0, k, n_kept = O.keys(plan, u, v, w, np.ones(M, np.complex64), np.ones(M, np.float32))
    s = np.float64(plan.N) * np.float64(plan.dl)
    x = (u.astype(np.longdouble) * np.longdouble(s) + np.longdouble(plan.N // 2)).astype(np.float64)
    y = (v.astype(np.longdouble) * np.longdouble(s) + np.longdouble(plan.N // 2)).astype(np.float64)
    ei0 = np.floor(x + 0.5).astype(np.int64)
    ej0 = np.floor(y + 0.5).astype(np.int64)
    inv_dw = np.float64(plan.Nw) / (np.float64(plan.w_max) - np.float64(plan.w_min))
    ek = np.floor((w.astype(np.float64) - plan.w_min) * inv_dw).astype(np.int64)
    ek = np.where((ek >= plan.Nw) & (w.astype(np.float64) <= plan.w_max), plan.Nw - 1, ek)
    h = (plan.support - 1) // 2
    keep = (ei0 >= h) & (ei0 <= plan.N - 1 - h) & (ej0 >= h) & (ej0 <= plan.N - 1 - h) & (ek >= 0) & (ek < plan.Nw)
    assert 0.3 < keep.mean() < 0.95
    assert n_kept == int(keep.sum())
    ekey = np.where(keep, (ek * plan.T + (ej0 >> 5)) * plan.T + (ei0 >> 5), plan.n_bins)
    assert np.array_equal(key, ekey.astype(np.uint32))
    assert np.array_equal(i0[keep], ei0[keep]) and np.array_equal(k[keep], ek[keep])


def test_stable_sort_three_ways():
    rng = np.random.default_rng(11)
    n_bins = 512
    key = rng.integers(0, n_bins + 1, 50000).astype(np.uint32)   # includes the sentinel n_bins
    key[rng.integers(0, key.size, 20000)] = 77                  # a hot bin
    perm = O.sort(key)
    perm2, bin_start = O.counting_sort(key, n_bins)
    perm3 = np.argsort(key, kind="stable").astype(np.uint32)
    assert np.array_equal(perm, perm2) and np.array_equal(perm, perm3)
    assert np.array_equal(bin_start, np.searchsorted(key[perm], np.arange(n_bins + 2), side="left").astype(np.uint64))
    assert key[perm[-1]] == n_bins    # the sentinel sorts last


def test_sort_cells_hand_case():
    """D4' order written out by hand: N = 64 (2 x 2 tiles), visibilities given by (i0, j0, k); k < 0 = dropped.
    Expected: plane first, then tile row, tile column, row in tile, column in tile, then input index."""
    #            idx: 0   1   2   3   4   5   6   7   8
    i0 = np.array([40,  5,  5, 33,  5, -1,  6,  5, 40], np.int32)
    j0 = np.array([ 3,  3, 35,  3,  3, -1,  3,  2,  3], np.int32)
    k = np.array([ 0,  1,  0,  0,  0, -1,  0,  0,  0], np.int32)
    # plane 0: tile (row 0, col 0): (j0 2, i0 5) idx 7; (3, 5) idx 4; (3, 6) idx 6
    #          tile (row 0, col 1): (3, 33) idx 3; (3, 40) idx 0, 8 (input order)
    #          tile (row 1, col 0): (35, 5) idx 2
    # plane 1: idx 1; dropped: idx 5
    assert list(O.sort_cells(i0, j0, k)) == [7, 4, 6, 3, 0, 8, 2, 1, 5]
    # col_drop = 1: columns 4|5 and 6|7 merge: (3,5) idx 4 and (3,6) idx 6 stay apart, (3,4)/(3,5) would merge
    i0b = np.array([5, 4, 7, 6], np.int32)
    z = np.zeros(4, np.int32)
    assert list(O.sort_cells(i0b, z + 3, z, col_drop=1)) == [0, 1, 2, 3]      # {5,4} tie -> input order, then {7,6}
    assert list(O.sort_cells(i0b, z + 3, z, col_drop=0)) == [1, 0, 3, 2]


def test_sort_cells_properties():
    """D4' on random inputs: a refinement of the D4 order (sorted by (plane, tile) key), lexicographic inside a
    tile, equal nearest cells contiguous and in input order, dropped visibilities last in input order; and
    the same permutation as numpy's lexsort over the same tuple."""
    rng = np.random.default_rng(3)
    for N, Nw in ((512, 16), (2048, 4)):
        plan = O.Plan(N=N, Nw=Nw, support=9, sigma=1.3, w_min=-50.0, w_max=50.0, dl=0.5 / N)
        M = 30000
        du = 1.0 / (N * plan.dl)
        u = rng.uniform(-0.52 * N * du, 0.52 * N * du, M).astype(np.float32)
        v = rng.uniform(-0.52 * N * du, 0.52 * N * du, M).astype(np.float32)
        u[:4000] = rng.uniform(40 * du, 60 * du, 4000).astype(np.float32)    # a dense patch: real runs
        v[:4000] = rng.uniform(40 * du, 60 * du, 4000).astype(np.float32)
        w = rng.uniform(-55, 55, M).astype(np.float32)
        key, i0, j0, k, n_kept = O.keys(plan, u, v, w, np.ones(M, np.complex64), np.ones(M, np.float32))
        perm = O.sort_cells(i0, j0, k).astype(np.int64)
        assert sorted(perm.tolist()) == list(range(M)) and 0 < n_kept < M
        kept, drop = perm[:n_kept], perm[n_kept:]
        assert np.all(k[kept] >= 0) and np.all(k[drop] < 0) and np.all(np.diff(drop) > 0)
        assert np.all(np.diff(key[perm].astype(np.int64)) >= 0)              # still sorted by the D4 tile key
        cell = (j0[kept].astype(np.int64) & 31) * 32 + (i0[kept] & 31)
        same_tile = np.diff(key[kept].astype(np.int64)) == 0
        assert np.all(np.diff(cell)[same_tile] >= 0)                          # lexicographic (row, column) in a tile
        full = (k[kept].astype(np.int64) * N + j0[kept]) * N + i0[kept]
        same_cell = np.diff(full) == 0
        assert np.all(np.diff(kept)[same_cell] > 0)                           # stable
        assert len(np.unique(full)) == 1 + int((~same_cell).sum())            # equal cells are contiguous
        big = np.where(k < 0, 1 << 40, 0).astype(np.int64)
        ref = np.lexsort((np.arange(M), i0 & 31, j0 & 31, i0 >> 5, j0 >> 5, k.astype(np.int64) + big))
        assert np.array_equal(perm, ref)
        # col_drop = 2: columns are compared in groups of four
        perm2 = O.sort_cells(i0, j0, k, col_drop=2).astype(np.int64)
        ref2 = np.lexsort((np.arange(M), (i0 & 31) >> 2, j0 & 31, i0 >> 5, j0 >> 5, k.astype(np.int64) + big))
        assert np.array_equal(perm2, ref2)


# ------------------------------------------------------------------------------------------------
# gridding
# ------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,sigma", [(7, 1.0), (9, 1.3)])
def test_single_visibility_footprint(S, sigma):
    plan = O.Plan(N=64, Nw=2, support=S, sigma=sigma, w_min=-1.0, w_max=1.0, dl=0.3 / 64)
    s = plan.N * plan.dl
    u = np.array([3.3 / s], np.float32)
    v = np.array([-7.8 / s], np.float32)
    w = np.array([0.5], np.float32)
    vis = np.array([1.5 - 0.25j], np.complex64)
    wt = np.array([0.75], np.float32)
    g = O.grid(plan, u, v, w, vis, wt)
    x = float(u[0]) * s + 32
    y = float(v[0]) * s + 32
    i0, j0, h = int(math.floor(x + 0.5)), int(math.floor(y + 0.5)), (S - 1) // 2
    exp = np.zeros((2, 64, 64), np.complex128)
    val = complex(vis[0]) * float(wt[0])
    for j in range(j0 - h, j0 + h + 1):
        for i in range(i0 - h, i0 + h + 1):
            exp[1, j, i] = val * math.exp(-((i - x) ** 2) / (2 * sigma ** 2)) * math.exp(-((j - y) ** 2) / (2 * sigma ** 2))
    assert np.count_nonzero(g) == S * S
    np.testing.assert_allclose(g, exp, rtol=1e-12, atol=1e-15)


@pytest.mark.parametrize("S,sigma", [(7, 1.0), (9, 1.3)])
def test_grid_sum_invariant_and_c0(S, sigma):
    rng = np.random.default_rng(3)
    plan = O.Plan(N=128, Nw=4, support=S, sigma=sigma, w_min=-50.0, w_max=50.0, dl=0.2 / 128)
    M = 5000
    u, v, w = _rand_vis(rng, M, plan.N, 0.2, -60, 60)     # some w out of range -> dropped
    vis = (rng.normal(size=M) + 1j * rng.normal(size=M)).astype(np.complex64)
    wt = rng.uniform(0.5, 1.0, M).astype(np.float32)
    g = O.grid(plan, u, v, w, vis, wt)
    _, i0, j0, k, n_kept = O.keys(plan, u, v, w, vis, wt)
    assert 0 < n_kept < M
    keep = k >= 0
    s = plan.N * plan.dl
    x = u.astype(np.float64) * s + plan.N // 2
    y = v.astype(np.float64) * s + plan.N // 2
    h = (S - 1) // 2
    a = np.arange(-h, h + 1)
    sx = np.exp(-((i0[:, None] + a[None, :] - x[:, None]) ** 2) / (2 * sigma ** 2)).sum(1)
    sy = np.exp(-((j0[:, None] + a[None, :] - y[:, None]) ** 2) / (2 * sigma ** 2)).sum(1)
    val = vis.astype(np.complex128) * wt.astype(np.float64)
    expected = (val * sx * sy)[keep].sum()
    assert abs(g.sum() - expected) <= 1e-12 * abs(expected)
    # per-plane sums too (a wrong plane index would move mass between planes)
    for kk in range(plan.Nw):
        e = (val * sx * sy)[k == kk].sum()
        assert abs(g[kk].sum() - e) <= 1e-11 * max(1.0, abs(e))
    # the mean tap sum over uniform offsets tends to c0 = integral of the truncated kernel (D8)
    c0 = O.taper(plan.N, S, sigma)[plan.N // 2]
    c0_quad = integrate.quad(lambda d: math.exp(-d * d / (2 * sigma ** 2)), -(h + 0.5), h + 0.5, epsabs=1e-14)[0]
    assert abs(c0 - c0_quad) < 1e-12
    assert abs(sx[keep].mean() - c0) < 5e-3 * c0


def test_taper_shape_is_gaussian_transform():
    N, S, sigma = 64, 7, 1.0
    t = O.taper(N, S, sigma)
    for p in (0, 5, 17, 32, 40, 63):
        nu = (p - N // 2) / N
        ft = integrate.quad(lambda d: math.exp(-d * d / (2 * sigma ** 2)) * math.cos(2 * math.pi * nu * d),
                            -40, 40, epsabs=1e-13, limit=400)[0]
        assert abs(t[p] / t[N // 2] - ft / (sigma * math.sqrt(2 * math.pi))) < 1e-10


# ------------------------------------------------------------------------------------------------
# plane transform (own FFT)
# ------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("N", [16, 32])
def test_fft_against_literal_double_sum(N):
    rng = np.random.default_rng(N)
    G = rng.normal(size=(N, N)) + 1j * rng.normal(size=(N, N))
    P = O.plane_transform(G)
    L = O.plane_transform_literal(G)
    assert np.max(np.abs(P - L)) <= 1e-12 * np.max(np.abs(L))
    # the literal sum itself against a numpy restatement of D7
    c = N // 2
    idx = np.arange(N) - c
    E = np.exp(2j * np.pi * np.outer(idx, idx) / N)     # E[p, i]
    L2 = E @ G.T                                          # sum_i E[p,i] G[j,i] -> [p, j]
    L2 = (E @ L2.T)                                       # sum_j E[q,j] (.)[p->col] -> [q, p]
    assert np.max(np.abs(L - L2)) <= 1e-12 * np.max(np.abs(L2))


@pytest.mark.parametrize("N", [64, 256])
def test_fft_against_numpy_parseval_delta(N):
    rng = np.random.default_rng(N)
    G = rng.normal(size=(N, N)) + 1j * rng.normal(size=(N, N))
    P = O.plane_transform(G)
    ref = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(G))) * (N * N)
    assert np.max(np.abs(P - ref)) <= 1e-12 * np.max(np.abs(ref))
    assert abs(np.sum(np.abs(P) ** 2) - N * N * np.sum(np.abs(G) ** 2)) <= 1e-12 * N * N * np.sum(np.abs(G) ** 2)
    D = np.zeros((N, N), np.complex128)
    D[N // 2, N // 2] = 1.0
    np.testing.assert_allclose(O.plane_transform(D), np.ones((N, N)), atol=1e-13)
    # a delta one cell off centre gives the pure phase ramp exp(2 pi i (p - N/2)/N): pins the sign
    D[:] = 0
    D[N // 2, N // 2 + 1] = 1.0
    ramp = np.exp(2j * np.pi * (np.arange(N) - N // 2) / N)
    np.testing.assert_allclose(O.plane_transform(D), np.tile(ramp, (N, 1)), atol=1e-12)


# ------------------------------------------------------------------------------------------------
# w screen, plane sum, taper
# ------------------------------------------------------------------------------------------------

def test_nm1_and_plane_centres():
    for l, m in [(0.0, 0.0), (0.01, -0.02), (0.15, 0.15), (-0.3, 0.2), (1e-5, 0.0)]:
        ref = np.sqrt(np.longdouble(1) - np.longdouble(l) ** 2 - np.longdouble(m) ** 2) - np.longdouble(1)
        assert abs(O.nm1(l, m) - float(ref)) <= 1e-15
    plan = O.Plan(N=64, Nw=4, support=7, sigma=1.0, w_min=-10.0, w_max=30.0, dl=0.001)
    assert [O.plane_centre(plan, k) for k in range(4)] == [-5.0, 5.0, 15.0, 25.0]


def test_wcorrect_against_numpy_restatement():
    rng = np.random.default_rng(8)
    plan = O.Plan(N=32, Nw=3, support=7, sigma=1.0, w_min=-200.0, w_max=400.0, dl=0.5 / 32)
    P = rng.normal(size=(3, 32, 32)) + 1j * rng.normal(size=(3, 32, 32))
    img = O.wcorrect(plan, P)
    l = (np.arange(32) - 16) * plan.dl
    ll, mm = np.meshgrid(l, l)                # image[q][p]: p <-> l fastest, q <-> m
    nm1 = np.sqrt(1 - ll ** 2 - mm ** 2) - 1
    t = O.taper(32, 7, 1.0)
    acc = np.zeros((32, 32))
    for k in range(3):
        wk = -200.0 + (k + 0.5) * 200.0
        acc += (np.exp(2j * np.pi * wk * nm1) * P[k]).real
    ref = acc / np.outer(t, t)
    assert np.max(np.abs(img - ref)) <= 1e-11 * np.max(np.abs(ref))
    # at the centre pixel the screen is exactly 1 for every plane
    assert abs(img[16, 16] * t[16] ** 2 - P[:, 16, 16].real.sum()) < 1e-13


def test_centre_pixel_invariant():
    """image[N/2][N/2] t[N/2]^2 = Re sum of the whole mesh -- links gridder and imager with no FFT."""
    rng = np.random.default_rng(21)
    plan = O.Plan(N=64, Nw=4, support=7, sigma=1.0, w_min=-80.0, w_max=80.0, dl=0.2 / 64)
    M = 3000
    u, v, w = _rand_vis(rng, M, plan.N, 0.2, -80, 80)
    vis = (rng.normal(size=M) + 1j * rng.normal(size=M)).astype(np.complex64)
    wt = rng.uniform(0.5, 1.0, M).astype(np.float32)
    img = O.image(plan, u, v, w, vis, wt)
    g = O.grid(plan, u, v, w, vis, wt)
    t = O.taper(plan.N, plan.support, plan.sigma)
    lhs = img[32, 32] * t[32] ** 2
    assert abs(lhs - g.sum().real) <= 1e-12 * np.abs(g).sum()


def test_image_equals_stagewise_composition():
    """rick_oracle_image (streamed) == grid -> transform each plane -> wcorrect."""
    rng = np.random.default_rng(22)
    plan = O.Plan(N=64, Nw=3, support=9, sigma=1.3, w_min=-40.0, w_max=50.0, dl=0.4 / 64)
    M = 2000
    u, v, w = _rand_vis(rng, M, plan.N, 0.4, -40, 50)
    vis = (rng.normal(size=M) + 1j * rng.normal(size=M)).astype(np.complex64)
    wt = rng.uniform(0.5, 1.0, M).astype(np.float32)
    img = O.image(plan, u, v, w, vis, wt)
    g = O.grid(plan, u, v, w, vis, wt)
    P = np.stack([O.plane_transform(g[k]) for k in range(plan.Nw)])
    img2 = O.wcorrect(plan, P)
    assert np.array_equal(img, img2)


# ------------------------------------------------------------------------------------------------
# end to end: closed forms and the brute-force direct DFT
# ------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,sigma", [(7, 1.0), (9, 1.3)])
def test_phase_centre_source_gives_weight_sum(S, sigma):
    """BASELINE.json north_star: a unit source at the phase centre with unit weights gives a peak equal
    to the weight sum."""
    rng = np.random.default_rng(31)
    plan = O.Plan(N=128, Nw=8, support=S, sigma=sigma, w_min=-300.0, w_max=300.0, dl=0.2 / 128)
    M = 5000
    u, v, w = _rand_vis(rng, M, plan.N, 0.2, -300, 300)
    vis = np.ones(M, np.complex64)
    wt = np.ones(M, np.float32)
    img, n_kept, _ = O.image(plan, u, v, w, vis, wt, return_timing=True)
    assert n_kept == M
    q, p = np.unravel_index(np.argmax(img), img.shape)
    assert (q, p) == (64, 64)
    assert abs(img[64, 64] / M - 1.0) <= 1e-4


@pytest.mark.parametrize("S,sigma", [(7, 1.0), (9, 1.3)])
def test_offset_source_peaks_at_its_pixel(S, sigma):
    rng = np.random.default_rng(32)
    plan = O.Plan(N=128, Nw=8, support=S, sigma=sigma, w_min=-300.0, w_max=300.0, dl=0.4 / 128)
    M = 5000
    u, v, w = _rand_vis(rng, M, plan.N, 0.4, -300, 300)
    w = _snap_w(plan, w)
    q0, p0 = 64 + 21, 64 - 13           # q <-> m, p <-> l (layout convention of the ABI)
    l0, m0 = (p0 - 64) * plan.dl, (q0 - 64) * plan.dl
    vis = _point_vis(u, v, w, l0, m0)
    wt = rng.uniform(0.5, 1.0, M).astype(np.float32)
    img = O.image(plan, u, v, w, vis, wt)
    q, p = np.unravel_index(np.argmax(img), img.shape)
    assert (q, p) == (q0, p0)
    assert abs(img[q0, p0] / wt.astype(np.float64).sum() - 1.0) <= 5e-3


@pytest.mark.parametrize("S,sigma,N", [(7, 1.0, 64), (9, 1.3, 64), (7, 1.0, 32)])
def test_against_bruteforce_direct_dft(S, sigma, N):
    """Oracle vs the exact dirty image D* (includes the w (n - 1) term), w snapped to plane centres so
    that only the gridding-kernel error remains; wide field so that the w term matters."""
    rng = np.random.default_rng(41)
    fov = 0.6
    plan = O.Plan(N=N, Nw=8, support=S, sigma=sigma, w_min=-150.0, w_max=150.0, dl=fov / N)
    M = 400
    u, v, w = _rand_vis(rng, M, N, fov, -150, 150, margin=5.0)
    w = _snap_w(plan, w)
    vis = np.zeros(M, np.complex64)
    for amp, l0, m0 in [(1.0, 0.11, -0.07), (0.7, -0.13, 0.12), (1.6, 0.02, 0.05)]:
        vis = vis + _point_vis(u, v, w, l0, m0, amp)
    wt = rng.uniform(0.5, 1.0, M).astype(np.float32)
    img = O.image(plan, u, v, w, vis, wt)
    ref = O.direct_dft(plan, u, v, w, vis, wt)
    # the brute force itself, retyped in numpy for one pixel
    q, p = N // 2 + 5, N // 2 - 9
    l, m = (p - N // 2) * plan.dl, (q - N // 2) * plan.dl
    ph = 2 * np.pi * (u.astype(np.float64) * l + v.astype(np.float64) * m + w.astype(np.float64) * (math.sqrt(1 - l * l - m * m) - 1))
    one = ((vis.astype(np.complex128) * wt.astype(np.float64)) * np.exp(1j * ph)).real.sum()
    assert abs(ref[q, p] - one) < 1e-9 * np.abs(ref).max()
    inner = slice(N // 4, 3 * N // 4)
    peak = np.abs(ref[inner, inner]).max()
    err = np.abs(img - ref)[inner, inner].max() / peak
    assert err <= 5e-3, err
    # dropping the w term must be visibly worse (a sign or missing-term error in the screen fails here)
    flat = O.Plan(N=N, Nw=1, support=S, sigma=sigma, w_min=-150.0, w_max=150.0, dl=fov / N)
    img_flat = O.image(flat, u, v, w, vis, wt)
    assert np.abs(img_flat - ref)[inner, inner].max() / peak > 10 * err


def test_w_stacking_converges_with_planes():
    rng = np.random.default_rng(42)
    N, fov = 64, 0.6
    M = 400
    u, v, w = _rand_vis(rng, M, N, fov, -150, 150, margin=5.0)
    vis = _point_vis(u, v, w, 0.11, -0.07) + _point_vis(u, v, w, -0.13, 0.12, 0.7)
    wt = np.ones(M, np.float32)
    inner = slice(N // 4, 3 * N // 4)
    errs = []
    for Nw in (2, 8, 32, 128, 512):
        plan = O.Plan(N=N, Nw=Nw, support=7, sigma=1.0, w_min=-150.0, w_max=150.0, dl=fov / N)
        img = O.image(plan, u, v, w, vis, wt)
        ref = O.direct_dft(plan, u, v, w, vis, wt)
        errs.append(np.abs(img - ref)[inner, inner].max() / np.abs(ref[inner, inner]).max())
    # the nearest-plane error falls like 1/Nw down to the gridding-kernel floor (~2e-3, see the test above)
    assert errs[0] > errs[1] > errs[2] > errs[3] > errs[4], errs
    assert errs[4] <= 6e-3, errs


# ------------------------------------------------------------------------------------------------
# structural properties
# ------------------------------------------------------------------------------------------------

def _setup(seed, M=3000, N=64, Nw=6, fov=0.5, wlim=120.0):
    rng = np.random.default_rng(seed)
    plan = O.Plan(N=N, Nw=Nw, support=7, sigma=1.0, w_min=-wlim, w_max=wlim, dl=fov / N)
    u, v, w = _rand_vis(rng, M, N, fov, -wlim, wlim)
    vis = (rng.normal(size=M) + 1j * rng.normal(size=M)).astype(np.complex64)
    wt = rng.uniform(0.5, 1.0, M).astype(np.float32)
    return rng, plan, u, v, w, vis, wt


def test_linearity():
    rng, plan, u, v, w, vis1, wt = _setup(51)
    vis2 = (rng.normal(size=vis1.size) + 1j * rng.normal(size=vis1.size)).astype(np.complex64)
    # exact fp32 combinations so that the fp32 inputs themselves are linear
    a, b = 2.0, -0.5
    vis3 = (a * vis1.astype(np.complex128) + b * vis2.astype(np.complex128))
    vis3_32 = vis3.astype(np.complex64)
    i1, i2 = O.image(plan, u, v, w, vis1, wt), O.image(plan, u, v, w, vis2, wt)
    i3 = O.image(plan, u, v, w, vis3_32, wt)
    # account for the rounding of vis3 to fp32 by imaging the residual too
    res = (vis3 - vis3_32.astype(np.complex128)).astype(np.complex64)
    i3 = i3 + O.image(plan, u, v, w, res, wt)
    peak = np.abs(i3).max()
    assert np.abs(i3 - (a * i1 + b * i2)).max() <= 1e-10 * peak


def test_hermitian_symmetry():
    """(u,v,w,V) -> (-u,-v,-w,conj V) gives the same image when w_min = -w_max and nothing sits on a
    rounding tie or at the drop boundary (taps and the FFT mirror through the centre node N/2)."""
    rng, plan, u, v, w, vis, wt = _setup(52)
    img = O.image(plan, u, v, w, vis, wt)
    img2 = O.image(plan, -u, -v, -w, np.conj(vis), wt)
    assert np.abs(img - img2).max() <= 1e-11 * np.abs(img).max()


def test_input_order_invariance():
    rng, plan, u, v, w, vis, wt = _setup(53)
    perm = rng.permutation(u.size)
    img = O.image(plan, u, v, w, vis, wt)
    img2 = O.image(plan, u[perm], v[perm], w[perm], vis[perm], wt[perm])
    # summation order changes the mesh by rounding; the taper division amplifies that towards the image
    # corners, so the difference is compared before that division (gate B of DESIGN.md)
    t = O.taper(plan.N, plan.support, plan.sigma)
    tw = np.outer(t, t) / t[plan.N // 2] ** 2
    assert (np.abs(img - img2) * tw).max() <= 1e-13 * np.abs(img * tw).max()
    inner = slice(plan.N // 4, 3 * plan.N // 4)
    assert np.abs(img - img2)[inner, inner].max() <= 1e-13 * np.abs(img[inner, inner]).max()


def test_thread_count_independence():
    rng, plan, u, v, w, vis, wt = _setup(54, M=1500)
    n = O.threads()
    try:
        O.set_threads(1)
        a = O.image(plan, u, v, w, vis, wt)
        O.set_threads(max(2, n))
        b = O.image(plan, u, v, w, vis, wt)
    finally:
        O.set_threads(n)
    assert np.array_equal(a, b)


def test_dropped_visibilities_do_not_contribute():
    rng, plan, u, v, w, vis, wt = _setup(55, M=500)
    # push 100 visibilities off the mesh / out of the w range / to NaN
    u2, w2, vis2 = u.copy(), w.copy(), vis.copy()
    u2[:40] = 1e6
    w2[40:80] = 1e4
    vis2[80:100] = np.nan
    img = O.image(plan, u2, v, w2, vis2, wt)
    img_ref = O.image(plan, u[100:], v[100:], w[100:], vis[100:], wt[100:])
    assert np.array_equal(img, img_ref)
    assert np.all(np.isfinite(img))
    # empty input -> zero image
    e = np.zeros(0, np.float32)
    z = O.image(plan, e, e, e, np.zeros(0, np.complex64), e)
    assert np.all(z == 0.0)


# ------------------------------------------------------------------------------------------------
# Kaiser-Bessel kernel (D6-KB: the kernel of the paper's own tests)
# ------------------------------------------------------------------------------------------------

KB = dict(kernel="kb", beta=2.34 * 7)


def _kb(d, a_t, beta):
    from scipy import special
    return special.i0(beta * np.sqrt(np.clip(1.0 - (np.asarray(d, np.float64) / a_t) ** 2, 0.0, None))) / special.i0(beta)


def test_kb_bessel_series_against_scipy():
    from scipy import special
    for x in (0.0, 1e-3, 0.7, 3.75, 9.0, 16.38, 21.06, 40.0):
        assert abs(O.bessel_i0(x) / special.i0(x) - 1.0) < 5e-15


@pytest.mark.parametrize("S,beta", [(7, 2.34 * 7), (9, 2.34 * 9), (5, 9.0)])
def test_kb_footprint_taper_and_tap_sum(S, beta):
    """Single-visibility footprint against the window typed with scipy's I0; the taper against numerical
    integration of the window (it is its exact transform); tap sums average to the taper's centre value."""
    h, a_t = (S - 1) // 2, (S - 1) // 2 + 0.5
    plan = O.Plan(N=64, Nw=2, support=S, sigma=1.0, w_min=-1.0, w_max=1.0, dl=0.3 / 64, kernel="kb", beta=beta)
    s = plan.N * plan.dl
    u = np.array([3.3 / s], np.float32)
    v = np.array([-7.8 / s], np.float32)
    g = O.grid(plan, u, v, np.array([0.5], np.float32), np.array([1.5 - 0.25j], np.complex64), np.array([0.75], np.float32))
    x, y = float(u[0]) * s + 32, float(v[0]) * s + 32
    i0, j0 = int(math.floor(x + 0.5)), int(math.floor(y + 0.5))
    exp = np.zeros((2, 64, 64), np.complex128)
    ii, jj = np.arange(i0 - h, i0 + h + 1), np.arange(j0 - h, j0 + h + 1)
    exp[1, j0 - h:j0 + h + 1, i0 - h:i0 + h + 1] = (1.5 - 0.25j) * 0.75 * np.outer(_kb(jj - y, a_t, beta), _kb(ii - x, a_t, beta))
    np.testing.assert_allclose(g, exp, rtol=1e-12, atol=1e-15)
    # the Gaussian oracle is untouched by the selection (state is set per call)
    g0 = O.grid(O.Plan(N=64, Nw=2, support=S, sigma=1.0, w_min=-1.0, w_max=1.0, dl=0.3 / 64), u, v,
                np.array([0.5], np.float32), np.array([1.0], np.complex64), np.array([1.0], np.float32))
    assert abs(g0[1, j0, i0] - math.exp(-((i0 - x) ** 2 + (j0 - y) ** 2) / 2.0)) < 1e-14
    N = 256
    t = O.taper(N, S, 1.0, "kb", beta)
    for p in (N // 2, N // 2 + 37, 11, 0):
        nu = (p - N // 2) / N
        val = integrate.quad(lambda d: float(_kb(d, a_t, beta)) * math.cos(2 * math.pi * nu * d), -a_t, a_t,
                             epsabs=1e-13, epsrel=1e-13, limit=400)[0]
        assert abs(val - t[p]) < 1e-11 * t[N // 2]
    rng = np.random.default_rng(8)
    off = rng.uniform(-0.5, 0.5, 20000)
    sums = _kb(off[:, None] + np.arange(-h, h + 1)[None, :], a_t, beta).sum(1)
    assert abs(sums.mean() - t[N // 2]) < 5e-3 * t[N // 2]


def test_kb_closed_forms_and_bruteforce():
    """Same end-to-end pins as for the Gaussian: phase-centre source -> weight sum; against the exact dirty
    image on a tiny wide-field case (the Kaiser-Bessel window aliases less: a tighter bound holds)."""
    rng = np.random.default_rng(31)
    plan = O.Plan(N=128, Nw=8, support=7, sigma=1.0, w_min=-300.0, w_max=300.0, dl=0.2 / 128, **KB)
    M = 5000
    u, v, w = _rand_vis(rng, M, plan.N, 0.2, -300, 300)
    img, n_kept, _ = O.image(plan, u, v, w, np.ones(M, np.complex64), np.ones(M, np.float32), return_timing=True)
    assert n_kept == M and np.unravel_index(np.argmax(img), img.shape) == (64, 64)
    assert abs(img[64, 64] / M - 1.0) <= 1e-4
    N, fov = 64, 0.6
    plan = O.Plan(N=N, Nw=8, support=7, sigma=1.0, w_min=-150.0, w_max=150.0, dl=fov / N, **KB)
    M = 400
    rng = np.random.default_rng(41)
    u, v, w = _rand_vis(rng, M, N, fov, -150, 150, margin=5.0)
    w = _snap_w(plan, w)
    vis = np.zeros(M, np.complex64)
    for amp, l0, m0 in [(1.0, 0.11, -0.07), (0.7, -0.13, 0.12), (1.6, 0.02, 0.05)]:
        vis = vis + _point_vis(u, v, w, l0, m0, amp)
    wt = rng.uniform(0.5, 1.0, M).astype(np.float32)
    img = O.image(plan, u, v, w, vis, wt)
    ref = O.direct_dft(plan, u, v, w, vis, wt)
    inner = slice(N // 4, 3 * N // 4)
    err = np.abs(img - ref)[inner, inner].max() / np.abs(ref[inner, inner]).max()
    gauss = O.image(O.Plan(N=N, Nw=8, support=7, sigma=1.0, w_min=-150.0, w_max=150.0, dl=fov / N), u, v, w, vis, wt)
    err_g = np.abs(gauss - ref)[inner, inner].max() / np.abs(ref[inner, inner]).max()
    print(f"KB vs exact {err:.2e}; Gaussian vs exact {err_g:.2e}")
    assert err <= 1e-3 and err < err_g
