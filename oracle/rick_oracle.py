"""ctypes/numpy front end of the CPU oracle (oracle/rick_oracle.cpp).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It never imports paper_2411_07321_b200 (the CUDA path) and the CUDA path never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rick_oracle.cpp")
_LIB = os.path.join(_HERE, "librick_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no CUDA involved)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
               _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        f32p, f64p = C.POINTER(C.c_float), C.POINTER(C.c_double)
        u32p, i32p, u64p = C.POINTER(C.c_uint32), C.POINTER(C.c_int32), C.POINTER(C.c_uint64)
        geo = [C.c_int, C.c_int, C.c_int]
        L.rick_oracle_threads.restype = C.c_int
        L.rick_oracle_set_threads.argtypes = [C.c_int]
        L.rick_oracle_set_kernel.argtypes = [C.c_int, C.c_double]
        L.rick_oracle_bessel_i0.restype = C.c_double
        L.rick_oracle_bessel_i0.argtypes = [C.c_double]
        L.rick_oracle_keys.restype = C.c_longlong
        L.rick_oracle_keys.argtypes = geo + [C.c_double, C.c_double, C.c_double, C.c_longlong,
                                             f32p, f32p, f32p, f32p, f32p, u32p, i32p, i32p, i32p]
        L.rick_oracle_sort.argtypes = [C.c_longlong, u32p, u32p]
        L.rick_oracle_sort_cells.argtypes = [C.c_longlong, i32p, i32p, i32p, C.c_int, u32p]
        L.rick_oracle_counting_sort.argtypes = [C.c_longlong, u32p, C.c_uint32, u32p, u64p]
        L.rick_oracle_grid.argtypes = geo + [C.c_double] * 4 + [C.c_longlong, f32p, f32p, f32p, f32p, f32p, f64p]
        L.rick_oracle_plane_transform.argtypes = [C.c_int, f64p]
        L.rick_oracle_plane_transform_literal.argtypes = [C.c_int, f64p, f64p]
        L.rick_oracle_taper.argtypes = [C.c_int, C.c_int, C.c_double, f64p]
        L.rick_oracle_nm1.restype = C.c_double
        L.rick_oracle_nm1.argtypes = [C.c_double, C.c_double]
        L.rick_oracle_plane_centre.restype = C.c_double
        L.rick_oracle_plane_centre.argtypes = [C.c_int, C.c_double, C.c_double, C.c_int]
        L.rick_oracle_wcorrect.argtypes = geo + [C.c_double] * 4 + [f64p, f64p]
        L.rick_oracle_image.restype = C.c_longlong
        L.rick_oracle_image.argtypes = geo + [C.c_double] * 4 + [C.c_longlong, f32p, f32p, f32p, f32p, f32p, f64p, f64p]
        L.rick_oracle_direct_dft.argtypes = geo + [C.c_double] * 3 + [C.c_longlong, f32p, f32p, f32p, f32p, f32p, f64p]
        _lib = L
    return _lib


def _p(a: np.ndarray, ct):
    return a.ctypes.data_as(C.POINTER(ct))


@dataclass(frozen=True)
class Plan:
    """Arguments of rick_plan_create (BASELINE.json north_star (1)); plain numbers only."""
    N: int
    Nw: int
    support: int
    sigma: float
    w_min: float
    w_max: float
    dl: float
    kernel: str = "gauss"      # "gauss" (D6, BASELINE.json north_star) or "kb" (D6-KB, the paper's kernel)
    beta: float = 0.0          # Kaiser-Bessel shape parameter (kernel == "kb")

    @property
    def T(self) -> int:
        return self.N // 32

    @property
    def n_bins(self) -> int:
        return self.Nw * self.T * self.T


def _select(kernel: str = "gauss", beta: float = 0.0) -> None:
    """Set the oracle's process-wide gridding kernel (done before every call that grids or tapers)."""
    if kernel not in ("gauss", "kb"):
        raise ValueError(kernel)
    lib().rick_oracle_set_kernel(1 if kernel == "kb" else 0, float(beta))


def bessel_i0(x: float) -> float:
    return float(lib().rick_oracle_bessel_i0(float(x)))


def _inputs(u, v, w, vis, wt):
    u = np.ascontiguousarray(u, dtype=np.float32)
    v = np.ascontiguousarray(v, dtype=np.float32)
    w = np.ascontiguousarray(w, dtype=np.float32)
    vis = np.ascontiguousarray(vis, dtype=np.complex64)
    wt = np.ascontiguousarray(wt, dtype=np.float32)
    M = u.shape[0]
    assert v.shape == (M,) and w.shape == (M,) and vis.shape == (M,) and wt.shape == (M,)
    return u, v, w, vis, wt, M


def threads() -> int:
    return int(lib().rick_oracle_threads())


def set_threads(n: int) -> None:
    lib().rick_oracle_set_threads(int(n))


def keys(plan: Plan, u, v, w, vis, wt):
    """-> (key u32[M], i0 i32[M], j0 i32[M], k i32[M], n_kept)."""
    u, v, w, vis, wt, M = _inputs(u, v, w, vis, wt)
    key = np.empty(M, np.uint32)
    i0 = np.empty(M, np.int32)
    j0 = np.empty(M, np.int32)
    k = np.empty(M, np.int32)
    n = lib().rick_oracle_keys(plan.N, plan.Nw, plan.support, plan.w_min, plan.w_max, plan.dl, M,
                               _p(u, C.c_float), _p(v, C.c_float), _p(w, C.c_float),
                               _p(vis.view(np.float32), C.c_float), _p(wt, C.c_float),
                               _p(key, C.c_uint32), _p(i0, C.c_int32), _p(j0, C.c_int32), _p(k, C.c_int32))
    return key, i0, j0, k, int(n)


def sort_cells(i0: np.ndarray, j0: np.ndarray, k: np.ndarray, col_drop: int = 0) -> np.ndarray:
    """D4': stable order by (plane, tile row, tile column, row in tile, column in tile >> col_drop), dropped
    visibilities (k < 0) last; i0 / j0 / k as returned by keys().  -> perm u32[M] (rank -> input index)."""
    i0 = np.ascontiguousarray(i0, dtype=np.int32)
    j0 = np.ascontiguousarray(j0, dtype=np.int32)
    k = np.ascontiguousarray(k, dtype=np.int32)
    perm = np.empty(k.shape[0], np.uint32)
    lib().rick_oracle_sort_cells(k.shape[0], _p(i0, C.c_int32), _p(j0, C.c_int32), _p(k, C.c_int32), int(col_drop),
                                 _p(perm, C.c_uint32))
    return perm


def sort(key: np.ndarray) -> np.ndarray:
    key = np.ascontiguousarray(key, dtype=np.uint32)
    perm = np.empty(key.shape[0], np.uint32)
    lib().rick_oracle_sort(key.shape[0], _p(key, C.c_uint32), _p(perm, C.c_uint32))
    return perm


def counting_sort(key: np.ndarray, n_bins: int) -> Tuple[np.ndarray, np.ndarray]:
    key = np.ascontiguousarray(key, dtype=np.uint32)
    perm = np.empty(key.shape[0], np.uint32)
    bin_start = np.empty(n_bins + 2, np.uint64)
    lib().rick_oracle_counting_sort(key.shape[0], _p(key, C.c_uint32), n_bins, _p(perm, C.c_uint32),
                                    _p(bin_start, C.c_uint64))
    return perm, bin_start


def grid(plan: Plan, u, v, w, vis, wt) -> np.ndarray:
    """-> complex128 [Nw, N, N] (D6; un-modulated mesh)."""
    u, v, w, vis, wt, M = _inputs(u, v, w, vis, wt)
    g = np.empty((plan.Nw, plan.N, plan.N), np.complex128)
    _select(plan.kernel, plan.beta)
    lib().rick_oracle_grid(plan.N, plan.Nw, plan.support, plan.sigma, plan.w_min, plan.w_max, plan.dl, M,
                           _p(u, C.c_float), _p(v, C.c_float), _p(w, C.c_float),
                           _p(vis.view(np.float32), C.c_float), _p(wt, C.c_float),
                           _p(g.view(np.float64), C.c_double))
    return g


def plane_transform(plane: np.ndarray) -> np.ndarray:
    """D7 via the oracle's own radix-2 FFT; returns a new array."""
    out = np.array(plane, dtype=np.complex128, order="C", copy=True)
    N = out.shape[0]
    assert out.shape == (N, N) and N & (N - 1) == 0
    lib().rick_oracle_plane_transform(N, _p(out.view(np.float64), C.c_double))
    return out


def plane_transform_literal(plane: np.ndarray) -> np.ndarray:
    src = np.ascontiguousarray(plane, dtype=np.complex128)
    N = src.shape[0]
    out = np.empty_like(src)
    lib().rick_oracle_plane_transform_literal(N, _p(src.view(np.float64), C.c_double),
                                              _p(out.view(np.float64), C.c_double))
    return out


def taper(N: int, support: int, sigma: float, kernel: str = "gauss", beta: float = 0.0) -> np.ndarray:
    t = np.empty(N, np.float64)
    _select(kernel, beta)
    lib().rick_oracle_taper(N, support, sigma, _p(t, C.c_double))
    return t


def nm1(l: float, m: float) -> float:
    return float(lib().rick_oracle_nm1(l, m))


def plane_centre(plan: Plan, k: int) -> float:
    return float(lib().rick_oracle_plane_centre(plan.Nw, plan.w_min, plan.w_max, k))


def wcorrect(plan: Plan, planes: np.ndarray) -> np.ndarray:
    P = np.ascontiguousarray(planes, dtype=np.complex128)
    assert P.shape == (plan.Nw, plan.N, plan.N)
    img = np.empty((plan.N, plan.N), np.float64)
    _select(plan.kernel, plan.beta)
    lib().rick_oracle_wcorrect(plan.N, plan.Nw, plan.support, plan.sigma, plan.w_min, plan.w_max, plan.dl,
                               _p(P.view(np.float64), C.c_double), _p(img, C.c_double))
    return img


def image(plan: Plan, u, v, w, vis, wt, return_timing: bool = False):
    """The whole path D2-D8 -> float64 [N, N] image (and n_kept, stage seconds)."""
    u, v, w, vis, wt, M = _inputs(u, v, w, vis, wt)
    img = np.empty((plan.N, plan.N), np.float64)
    st = np.zeros(4, np.float64)
    _select(plan.kernel, plan.beta)
    n = lib().rick_oracle_image(plan.N, plan.Nw, plan.support, plan.sigma, plan.w_min, plan.w_max, plan.dl, M,
                                _p(u, C.c_float), _p(v, C.c_float), _p(w, C.c_float),
                                _p(vis.view(np.float32), C.c_float), _p(wt, C.c_float),
                                _p(img, C.c_double), _p(st, C.c_double))
    if return_timing:
        return img, int(n), dict(keys=st[0], grid=st[1], fft=st[2], wcorrect=st[3])
    return img


def direct_dft(plan: Plan, u, v, w, vis, wt) -> np.ndarray:
    """Brute-force exact dirty image D* over the kept visibilities (tiny inputs only)."""
    u, v, w, vis, wt, M = _inputs(u, v, w, vis, wt)
    img = np.empty((plan.N, plan.N), np.float64)
    lib().rick_oracle_direct_dft(plan.N, plan.Nw, plan.support, plan.w_min, plan.w_max, plan.dl, M,
                                 _p(u, C.c_float), _p(v, C.c_float), _p(w, C.c_float),
                                 _p(vis.view(np.float32), C.c_float), _p(wt, C.c_float), _p(img, C.c_double))
    return img
