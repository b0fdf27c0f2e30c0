"""Thin ctypes binding of librick_b200 (include/rick_b200.h): argument marshalling only.

PyTorch owns device memory and streams; every step of the hot path runs inside the library's CUDA
kernels (plus batched cuFFT for the plane transforms).  There is no CPU fallback: if the shared library
is missing or cannot be loaded, importing symbols from it raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import torch

from . import build as _build

RICK_C64, RICK_C128 = 0, 1
RICK_T_NAMES = ("bin", "zero", "grid", "fft", "wcorrect", "image", "keygen", "sort", "gather", "fft_rows", "fft_col_a")

_lib = None

EXPORTS = (
    "rick_plan_create", "rick_plan_set_dtype", "rick_plan_workspace_bytes", "rick_plan_destroy",
    "rick_plan_sort_layout", "rick_plan_set_fusion", "rick_plan_set_kernel", "rick_plan_rows_defined",
    "rick_bin", "rick_grid", "rick_fft_planes", "rick_wcorrect_accumulate", "rick_image",
    "rick_image_from_host", "rick_image_from_host_chunked", "rick_get_timings", "rick_launch_count", "rick_strerror",
    "rick_measure_fp32_rate", "rick_measure_random_read_rate", "rick_bin_static", "rick_plan_cells_defined",
)


class RickError(RuntimeError):
    pass


class _DeviceBuffers(C.Structure):
    _fields_ = [
        ("u", C.c_void_p), ("v", C.c_void_p), ("w", C.c_void_p), ("vis", C.c_void_p), ("weight", C.c_void_p),
        ("u_s", C.c_void_p), ("v_s", C.c_void_p), ("w_s", C.c_void_p), ("vis_s", C.c_void_p), ("weight_s", C.c_void_p),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
        ("grid", C.c_void_p),
        ("fft_work", C.c_void_p), ("fft_work_bytes", C.c_size_t),
        ("image", C.c_void_p),
        ("n_kept", C.c_void_p),
    ]


def library_path() -> str:
    return _build.LIB


def lib():
    """Load librick_b200.so (built in-tree by __graft_entry__.build()); fails loudly when absent."""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise RickError(f"{path} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                            "(the CUDA library is the only implementation; there is no fallback)")
        L = C.CDLL(path)
        vp, ll, sz, dbl, i = C.c_void_p, C.c_longlong, C.c_size_t, C.c_double, C.c_int
        L.rick_plan_create.argtypes = [i, i, i, dbl, dbl, dbl, dbl, C.POINTER(vp)]
        L.rick_plan_set_dtype.argtypes = [vp, i]
        L.rick_plan_workspace_bytes.argtypes = [vp, ll, C.POINTER(sz), C.POINTER(sz)]
        L.rick_plan_destroy.argtypes = [vp]
        L.rick_plan_set_fusion.argtypes = [vp, i]
        L.rick_plan_set_kernel.argtypes = [vp, i, dbl]
        L.rick_plan_rows_defined.argtypes = [vp, C.POINTER(ll)]
        L.rick_plan_cells_defined.argtypes = [vp, C.POINTER(ll)]
        L.rick_plan_sort_layout.argtypes = [vp, C.POINTER(i), C.POINTER(i), C.POINTER(i)]
        L.rick_bin.argtypes = [vp, ll] + [vp] * 5 + [vp] * 5 + [vp, vp, vp, vp, sz, vp, vp]
        L.rick_bin_static.argtypes = [vp, ll] + [vp] * 5 + [vp] * 5 + [vp, vp, vp, vp, vp]
        L.rick_grid.argtypes = [vp, vp, i, vp]
        L.rick_fft_planes.argtypes = [vp, vp, vp, sz, vp]
        L.rick_wcorrect_accumulate.argtypes = [vp, vp, vp, i, vp]
        L.rick_image.argtypes = [vp, vp, vp, i, vp]
        L.rick_image_from_host.argtypes = [vp, ll, vp, vp, vp, vp, vp, C.POINTER(_DeviceBuffers), vp, vp]
        L.rick_image_from_host_chunked.argtypes = [vp, ll, vp, vp, vp, vp, vp, C.POINTER(_DeviceBuffers), i, vp, vp]
        L.rick_get_timings.argtypes = [vp, C.POINTER(dbl), i]
        L.rick_launch_count.argtypes = [vp]
        L.rick_launch_count.restype = ll
        L.rick_measure_fp32_rate.argtypes = [C.POINTER(dbl), C.POINTER(dbl), C.POINTER(dbl), vp]
        L.rick_measure_random_read_rate.argtypes = [C.POINTER(dbl), vp]
        L.rick_strerror.argtypes = [i]
        L.rick_strerror.restype = C.c_char_p
        for name in EXPORTS:
            getattr(L, name)
        _lib = L
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise RickError(f"{what} failed: {lib().rick_strerror(rc).decode()} ({rc})")


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _stream(stream=None) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream


def _dev(t: torch.Tensor, dtype, n: Optional[int] = None, what: str = "tensor") -> torch.Tensor:
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise RickError(f"{what}: expected a contiguous CUDA tensor of {dtype}")
    if n is not None and t.numel() < n:
        raise RickError(f"{what}: needs at least {n} elements")
    return t


# ---- the C entry points, one Python function each ---------------------------------------------

def rick_plan_create(N: int, Nw: int, support: int, sigma: float, w_min: float, w_max: float, dl: float) -> int:
    h = C.c_void_p()
    _check(lib().rick_plan_create(N, Nw, support, sigma, w_min, w_max, dl, C.byref(h)), "rick_plan_create")
    return h.value


def rick_plan_set_dtype(plan: int, dtype: int) -> None:
    _check(lib().rick_plan_set_dtype(plan, dtype), "rick_plan_set_dtype")


def rick_plan_workspace_bytes(plan: int, M: int):
    a, b = C.c_size_t(), C.c_size_t()
    _check(lib().rick_plan_workspace_bytes(plan, M, C.byref(a), C.byref(b)), "rick_plan_workspace_bytes")
    return int(a.value), int(b.value)


def rick_plan_sort_layout(plan: int):
    """-> (key_bits, n_pass, cell_bits) of the sort key [D4']."""
    a, b, c = C.c_int(), C.c_int(), C.c_int()
    _check(lib().rick_plan_sort_layout(plan, C.byref(a), C.byref(b), C.byref(c)), "rick_plan_sort_layout")
    return int(a.value), int(b.value), int(c.value)


def rick_plan_set_fusion(plan: int, on: int) -> int:
    """Fused column transform: 0 off, 1 on, 2 on + row-occupancy tracking (rick_b200.h).  Returns the mode in
    force: 0 when the plan does not support fusion."""
    on = int(on)
    rc = lib().rick_plan_set_fusion(plan, on)
    if rc == -1 and on:      # RICK_EINVAL: dtype / N not supported by the fused kernel
        return 0
    _check(rc, "rick_plan_set_fusion")
    return on


def rick_plan_rows_defined(plan: int) -> int:
    """Fusion mode 2: mesh rows that held defined data at the last rick_fft_planes."""
    n = C.c_longlong()
    _check(lib().rick_plan_rows_defined(plan, C.byref(n)), "rick_plan_rows_defined")
    return int(n.value)


def rick_plan_cells_defined(plan: int) -> int:
    """Fusion mode 2: mesh cells that hold defined data (defined segments, or defined rows where rows are the unit)."""
    n = C.c_longlong()
    _check(lib().rick_plan_cells_defined(plan, C.byref(n)), "rick_plan_cells_defined")
    return int(n.value)


RICK_KERNEL_GAUSS, RICK_KERNEL_KB = 0, 1


def rick_plan_set_kernel(plan: int, kind: int, param: float = 0.0) -> None:
    """Gridding kernel: RICK_KERNEL_GAUSS (default) or RICK_KERNEL_KB with shape parameter beta = param."""
    _check(lib().rick_plan_set_kernel(plan, int(kind), float(param)), "rick_plan_set_kernel")


def rick_plan_destroy(plan: int) -> None:
    _check(lib().rick_plan_destroy(plan), "rick_plan_destroy")


def rick_bin(plan: int, M: int, u, v, w, vis, weight, u_s, v_s, w_s, vis_s, weight_s, workspace, n_kept,
             key_out=None, perm_out=None, bin_start_out=None, stream=None) -> None:
    f32, c64 = torch.float32, torch.complex64
    for t, dt, nm in ((u, f32, "u"), (v, f32, "v"), (w, f32, "w"), (vis, c64, "vis"), (weight, f32, "weight")):
        _dev(t, dt, M, nm)
    for t, dt, nm in ((u_s, f32, "u_s"), (v_s, f32, "v_s"), (w_s, f32, "w_s"), (vis_s, c64, "vis_s"),
                      (weight_s, f32, "weight_s")):
        if t is not None:        # all five None: no sorted copies (fp32 mesh; the gridder fetches records by index)
            _dev(t, dt, M, nm)
    _dev(workspace, torch.uint8, None, "workspace")
    _dev(n_kept, torch.int64, 1, "n_kept")
    if key_out is not None:
        _dev(key_out, torch.int32, M, "key_out")
    if perm_out is not None:
        _dev(perm_out, torch.int32, M, "perm_out")
    if bin_start_out is not None:
        _dev(bin_start_out, torch.int64, None, "bin_start_out")
    _check(lib().rick_bin(plan, M, _ptr(u), _ptr(v), _ptr(w), _ptr(vis), _ptr(weight), _ptr(u_s), _ptr(v_s),
                          _ptr(w_s), _ptr(vis_s), _ptr(weight_s), _ptr(key_out), _ptr(perm_out),
                          _ptr(bin_start_out), _ptr(workspace), workspace.numel(), _ptr(n_kept), _stream(stream)),
           "rick_bin")


RICK_BIN_STATIC_MAX_M = 262144


def rick_bin_static(plan: int, M: int, u, v, w, vis, weight, u_s, v_s, w_s, vis_s, weight_s, n_kept,
                    key_out=None, perm_out=None, bin_start_out=None, stream=None) -> None:
    """rick_bin with the library's static device scratch instead of a caller workspace: allocates nothing,
    M <= RICK_BIN_STATIC_MAX_M (RICK_ELIMIT beyond), calls that overlap on the GPU race (rick_b200.h)."""
    f32, c64 = torch.float32, torch.complex64
    for t, dt, nm in ((u, f32, "u"), (v, f32, "v"), (w, f32, "w"), (vis, c64, "vis"), (weight, f32, "weight")):
        _dev(t, dt, min(M, RICK_BIN_STATIC_MAX_M), nm)
    for t, dt, nm in ((u_s, f32, "u_s"), (v_s, f32, "v_s"), (w_s, f32, "w_s"), (vis_s, c64, "vis_s"),
                      (weight_s, f32, "weight_s")):
        if t is not None:
            _dev(t, dt, min(M, RICK_BIN_STATIC_MAX_M), nm)
    _dev(n_kept, torch.int64, 1, "n_kept")
    if key_out is not None:
        _dev(key_out, torch.int32, min(M, RICK_BIN_STATIC_MAX_M), "key_out")
    if perm_out is not None:
        _dev(perm_out, torch.int32, min(M, RICK_BIN_STATIC_MAX_M), "perm_out")
    if bin_start_out is not None:
        _dev(bin_start_out, torch.int64, None, "bin_start_out")
    _check(lib().rick_bin_static(plan, M, _ptr(u), _ptr(v), _ptr(w), _ptr(vis), _ptr(weight), _ptr(u_s), _ptr(v_s),
                                 _ptr(w_s), _ptr(vis_s), _ptr(weight_s), _ptr(key_out), _ptr(perm_out),
                                 _ptr(bin_start_out), _ptr(n_kept), _stream(stream)), "rick_bin_static")


def rick_grid(plan: int, grid: torch.Tensor, zero_first: bool = True, stream=None) -> None:
    if not (grid.is_cuda and grid.is_contiguous()):
        raise RickError("grid: expected a contiguous CUDA tensor")
    _check(lib().rick_grid(plan, _ptr(grid), 1 if zero_first else 0, _stream(stream)), "rick_grid")


def rick_fft_planes(plan: int, grid: torch.Tensor, fft_work: Optional[torch.Tensor], stream=None) -> None:
    nbytes = 0 if fft_work is None else fft_work.numel() * fft_work.element_size()
    _check(lib().rick_fft_planes(plan, _ptr(grid), _ptr(fft_work), nbytes, _stream(stream)), "rick_fft_planes")


def rick_wcorrect_accumulate(plan: int, grid: torch.Tensor, image: torch.Tensor, zero_first: bool = True,
                             stream=None) -> None:
    _dev(image, torch.float64, None, "image")
    _check(lib().rick_wcorrect_accumulate(plan, _ptr(grid), _ptr(image), 1 if zero_first else 0, _stream(stream)),
           "rick_wcorrect_accumulate")


def rick_image(plan: int, image_dev: torch.Tensor, out: torch.Tensor, stream=None) -> None:
    _dev(image_dev, torch.float64, None, "image_dev")
    if out.dtype != torch.float64 or not out.is_contiguous() or out.numel() < image_dev.numel():
        raise RickError("out: expected a contiguous float64 tensor of N*N elements")
    _check(lib().rick_image(plan, _ptr(image_dev), _ptr(out), 0 if out.is_cuda else 1, _stream(stream)), "rick_image")


def rick_get_timings(plan: int) -> Dict[str, float]:
    arr = (C.c_double * len(RICK_T_NAMES))()
    _check(lib().rick_get_timings(plan, arr, len(RICK_T_NAMES)), "rick_get_timings")
    return {n: float(arr[i]) for i, n in enumerate(RICK_T_NAMES)}


def rick_launch_count(plan: int) -> int:
    return int(lib().rick_launch_count(plan))


def rick_measure_fp32_rate():
    """-> (fp32 FMA TFLOP/s, 1e12 fp32 adds / s, packed-FMA TFLOP/s) measured on the current device."""
    a, b, c = C.c_double(), C.c_double(), C.c_double()
    _check(lib().rick_measure_fp32_rate(C.byref(a), C.byref(b), C.byref(c), _stream()), "rick_measure_fp32_rate")
    return float(a.value), float(b.value), float(c.value)


def rick_measure_random_read_rate() -> float:
    """-> 1e9 random 32-byte records read per second, measured on the current device (measurement helper)."""
    a = C.c_double()
    _check(lib().rick_measure_random_read_rate(C.byref(a), _stream()), "rick_measure_random_read_rate")
    return float(a.value)


# ---- buffer ownership helper (allocation + marshalling; no arithmetic) --------------------------

class Imager:
    """Owns the plan handle and the torch device buffers for one configuration and calls the C entry
    points in path order.  Nothing is computed in Python."""

    def __init__(self, N: int, Nw: int, support: int, sigma: float, w_min: float, w_max: float, dl: float,
                 dtype: str = "c64", M_max: int = 0, device="cuda", fused: int = 0,
                 kernel: str = "gauss", beta: float = 0.0, alloc_mesh: bool = True,
                 sorted_outputs: Optional[bool] = None):
        if not torch.cuda.is_available():
            raise RickError("librick_b200 needs a CUDA device (no CPU fallback)")
        self.device = torch.device(device)
        self.N, self.Nw, self.support = N, Nw, support
        self.dtype = RICK_C128 if dtype == "c128" else RICK_C64
        self.cdtype = torch.complex128 if dtype == "c128" else torch.complex64
        with torch.cuda.device(self.device):
            self.plan = rick_plan_create(N, Nw, support, sigma, w_min, w_max, dl)
            rick_plan_set_dtype(self.plan, self.dtype)
            self.fused = rick_plan_set_fusion(self.plan, int(fused)) if fused else 0
            if kernel == "kb":
                rick_plan_set_kernel(self.plan, RICK_KERNEL_KB, beta)
            elif kernel != "gauss":
                raise RickError(f"unknown gridding kernel {kernel!r}")
        # sorted SoA copies of the kept visibilities (an output of rick_bin): the fp64 gridder reads them; on the
        # fp32 mesh they are optional, and without them rick_bin gathers nothing (indirect mode, rick_b200.h)
        self.sorted_outputs = (dtype == "c128") if sorted_outputs is None else bool(sorted_outputs)
        if dtype == "c128" and not self.sorted_outputs:
            raise RickError("the fp64 mesh needs the sorted outputs of rick_bin")
        self.M_max = 0
        # alloc_mesh = False: a binning-only helper (rick_bin needs neither the mesh nor the image)
        self.grid = torch.empty((Nw, N, N) if alloc_mesh else (0,), dtype=self.cdtype, device=self.device)
        self.image = torch.empty((N, N) if alloc_mesh else (0,), dtype=torch.float64, device=self.device)
        self.n_kept = torch.zeros(1, dtype=torch.int64, device=self.device)
        _, fft_bytes = rick_plan_workspace_bytes(self.plan, 0)
        self.fft_work = torch.empty(fft_bytes, dtype=torch.uint8, device=self.device) if fft_bytes else None
        self.sorted = None
        self.workspace = None
        self.staging = None
        self.reserve(M_max)

    def reserve(self, M: int) -> None:
        if M <= self.M_max and self.sorted is not None:
            return
        m = max(int(M), 1)
        d = self.device
        ms = m if self.sorted_outputs else 0
        self.sorted = dict(u=torch.empty(ms, dtype=torch.float32, device=d), v=torch.empty(ms, dtype=torch.float32, device=d),
                           w=torch.empty(ms, dtype=torch.float32, device=d), vis=torch.empty(ms, dtype=torch.complex64, device=d),
                           weight=torch.empty(ms, dtype=torch.float32, device=d))
        bin_bytes, _ = rick_plan_workspace_bytes(self.plan, m)
        self.workspace = torch.empty(bin_bytes, dtype=torch.uint8, device=d)
        self.staging = None
        self.M_max = m

    def close(self) -> None:
        if self.plan:
            rick_plan_destroy(self.plan)
            self.plan = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # path steps
    def bin(self, u, v, w, vis, weight, key_out=None, perm_out=None, bin_start_out=None) -> None:
        M = int(u.numel())
        self.reserve(M)
        s = self.sorted if self.sorted_outputs else dict(u=None, v=None, w=None, vis=None, weight=None)
        rick_bin(self.plan, M, u, v, w, vis, weight, s["u"], s["v"], s["w"], s["vis"], s["weight"], self.workspace,
                 self.n_kept, key_out=key_out, perm_out=perm_out, bin_start_out=bin_start_out)

    def grid_(self, zero_first: bool = True) -> None:
        rick_grid(self.plan, self.grid, zero_first)

    def fft(self) -> None:
        rick_fft_planes(self.plan, self.grid, self.fft_work)

    def wcorrect(self, zero_first: bool = True) -> None:
        rick_wcorrect_accumulate(self.plan, self.grid, self.image, zero_first)

    def run(self, u, v, w, vis, weight) -> torch.Tensor:
        """bin -> grid -> FFT -> w-correct on device-resident inputs; returns the device image."""
        self.bin(u, v, w, vis, weight)
        self.grid_(True)
        self.fft()
        self.wcorrect(True)
        return self.image

    def run_from_host(self, u, v, w, vis, weight, image_host: torch.Tensor, chunks: int = 1) -> torch.Tensor:
        """rick_image_from_host (chunks == 1) / rick_image_from_host_chunked: host (pinned) inputs -> host
        image, copies included; with chunks > 1 the copies of one slice overlap the gridding of the last."""
        M = int(u.numel())
        self.reserve(M)
        if self.staging is None:
            d = self.device
            m = self.M_max
            self.staging = dict(u=torch.empty(m, dtype=torch.float32, device=d), v=torch.empty(m, dtype=torch.float32, device=d),
                                w=torch.empty(m, dtype=torch.float32, device=d), vis=torch.empty(m, dtype=torch.complex64, device=d),
                                weight=torch.empty(m, dtype=torch.float32, device=d))
        for t in (u, v, w, vis, weight, image_host):
            if t.is_cuda or not t.is_contiguous():
                raise RickError("run_from_host: host tensors expected")
        g = self.staging
        s = self.sorted if self.sorted_outputs else dict(u=None, v=None, w=None, vis=None, weight=None)
        b = _DeviceBuffers(
            _ptr(g["u"]), _ptr(g["v"]), _ptr(g["w"]), _ptr(g["vis"]), _ptr(g["weight"]),
            _ptr(s["u"]), _ptr(s["v"]), _ptr(s["w"]), _ptr(s["vis"]), _ptr(s["weight"]),
            _ptr(self.workspace), self.workspace.numel(), _ptr(self.grid),
            _ptr(self.fft_work), 0 if self.fft_work is None else self.fft_work.numel(),
            _ptr(self.image), _ptr(self.n_kept))
        if chunks > 1:
            _check(lib().rick_image_from_host_chunked(self.plan, M, _ptr(u), _ptr(v), _ptr(w), _ptr(vis), _ptr(weight),
                                                      C.byref(b), int(chunks), _ptr(image_host), _stream()),
                   "rick_image_from_host_chunked")
        else:
            _check(lib().rick_image_from_host(self.plan, M, _ptr(u), _ptr(v), _ptr(w), _ptr(vis), _ptr(weight),
                                              C.byref(b), _ptr(image_host), _stream()), "rick_image_from_host")
        return image_host

    def timings(self) -> Dict[str, float]:
        return rick_get_timings(self.plan)

    def launches(self) -> int:
        return rick_launch_count(self.plan)
