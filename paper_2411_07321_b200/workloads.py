"""Seeded synthetic visibility workloads (input data only -- none of the imaging method lives here).

These stand in for the paper's LOFAR HBA measurement sets (Table 1; mesh
shapes Table 2), which are not available.  The five configurations are the ones
BASELINE.json `configs` names; every free choice is listed in DESIGN.md "Input recipe".

What is generated:
  * antenna ENU positions -> equatorial XYZ -> (u, v, w) tracks in wavelengths (textbook synthesis,
    Taylor et al. 1999, cited at PAPER.md line 24), time-major row order,
    channel innermost;
  * model visibilities of point sources through the measurement equation, Eq. 1 (line 48),
    plus Gaussian noise, and a weight per measurement.

This module is shared by the CUDA path's tests/bench and by the oracle's tests as *data*.  It imports
neither of them.  All randomness is counter based (splitmix64 of (seed, stream, index)), evaluated
with torch integer ops so that the same code runs on the CPU (tests) and on the GPU (large configs).
Arrays are produced once and the same arrays are handed to both sides.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Dict, Optional, Tuple

import torch

BASE_SEED = 241107321
C_LIGHT = 299792458.0

# RNG streams
_STREAM_ANT, _STREAM_SRC, _STREAM_NOISE, _STREAM_WEIGHT, _STREAM_HOT = 1, 2, 3, 4, 5


def _s64(x: int) -> int:
    """Wrap an unsigned 64-bit constant into Python's view of a signed int64."""
    x &= (1 << 64) - 1
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLD = _s64(0x9E3779B97F4A7C15)
_M1 = _s64(0xBF58476D1CE4E5B9)
_M2 = _s64(0x94D049BB133111EB)
_K_SEED = 0xD1342543DE82EF95
_K_STREAM = 0xA24BAED4963EE407


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right of an int64 tensor."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix64(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _M1
    z = (z ^ _lsr(z, 27)) * _M2
    return z ^ _lsr(z, 31)


def rng_uniform(seed: int, stream: int, index: torch.Tensor) -> torch.Tensor:
    """Counter-based U[0,1) in float64; `index` is an int64 tensor of counters."""
    base = _s64(seed * _K_SEED + stream * _K_STREAM)
    z = index * _GOLD + base
    z = _mix64(_mix64(z) + _GOLD)
    return _lsr(z, 11).to(torch.float64) * (1.0 / 9007199254740992.0)


def rng_normal(seed: int, stream: int, index: torch.Tensor) -> torch.Tensor:
    """Counter-based N(0,1) (Box-Muller on counters 2i, 2i+1)."""
    u1 = rng_uniform(seed, stream, index * 2)
    u2 = rng_uniform(seed, stream, index * 2 + 1)
    return torch.sqrt(-2.0 * torch.log1p(-u1)) * torch.cos((2.0 * math.pi) * u2)


@dataclass(frozen=True)
class Config:
    """One BASELINE.json configuration: the data recipe plus the plan parameters it is imaged with."""
    name: str
    M: int                       # visibilities
    n_ant_core: int
    n_ant_outer: int
    core_sigma_m: float          # E,N ~ N(0, core_sigma)
    core_up_sigma_m: float       # U ~ N(0, .) (0 for a flat core)
    outer_rmin_m: float
    outer_rmax_m: float
    n_times: int
    ha_range_h: float            # hour angle in +-ha_range_h
    freqs_hz: Tuple[float, ...]
    n_src: int
    flux: str                    # "uniform" (U(0.5,2)) or "powerlaw"
    lm_max: float
    noise_sigma: float
    weights: str                 # "unit" or "uniform" (U(0.5,1))
    hotspot_frac: float = 0.0    # fraction of rows replaced by a dense uv disc
    hotspot_radius_lambda: float = 200.0
    hotspot_w_lambda: float = 100.0
    # plan
    N: int = 256
    Nw: int = 8
    support: int = 7
    sigma: float = 1.0
    dtype: str = "c128"          # mesh dtype: "c64" | "c128"
    fov: float = 0.2             # N * dl
    dec_deg: float = 50.0
    lat_deg: float = 52.9
    seed: int = BASE_SEED

    @property
    def dl(self) -> float:
        return self.fov / self.N

    @property
    def n_bl(self) -> int:
        n = self.n_ant_core + self.n_ant_outer
        return n * (n - 1) // 2

    @property
    def n_ch(self) -> int:
        return len(self.freqs_hz)


def _chan(lo_mhz: float, hi_mhz: float, n: int) -> Tuple[float, ...]:
    if n == 1:
        return (lo_mhz * 1e6,)
    return tuple((lo_mhz + (hi_mhz - lo_mhz) * c / (n - 1)) * 1e6 for c in range(n))


CONFIGS: Dict[str, Config] = {
    # BASELINE.json configs[0]
    "tiny": Config(name="tiny", M=100_000, n_ant_core=16, n_ant_outer=0, core_sigma_m=500.0,
                   core_up_sigma_m=500.0, outer_rmin_m=0.0, outer_rmax_m=0.0, n_times=834,
                   ha_range_h=2.0, freqs_hz=(150e6,), n_src=3, flux="uniform", lm_max=0.05,
                   noise_sigma=0.01, weights="unit", N=256, Nw=8, support=7, sigma=1.0,
                   dtype="c128", fov=0.2),
    # BASELINE.json configs[1]
    "10M": Config(name="10M", M=10_000_000, n_ant_core=42, n_ant_outer=20, core_sigma_m=300.0,
                  core_up_sigma_m=0.0, outer_rmin_m=1e3, outer_rmax_m=50e3, n_times=5289,
                  ha_range_h=4.0, freqs_hz=(144e6,), n_src=50, flux="powerlaw", lm_max=0.05,
                  noise_sigma=0.01, weights="uniform", N=2048, Nw=32, support=7, sigma=1.0,
                  dtype="c64", fov=0.2),
    # BASELINE.json configs[2]
    "100M": Config(name="100M", M=100_000_000, n_ant_core=42, n_ant_outer=20, core_sigma_m=300.0,
                   core_up_sigma_m=0.0, outer_rmin_m=1e3, outer_rmax_m=50e3, n_times=6611,
                   ha_range_h=4.0, freqs_hz=_chan(120.0, 168.0, 8), n_src=50, flux="powerlaw",
                   lm_max=0.15, noise_sigma=0.01, weights="uniform", N=4096, Nw=64, support=7,
                   sigma=1.0, dtype="c128", fov=0.6),
    # BASELINE.json configs[3]
    "500M": Config(name="500M", M=500_000_000, n_ant_core=42, n_ant_outer=20, core_sigma_m=300.0,
                   core_up_sigma_m=0.0, outer_rmin_m=1e3, outer_rmax_m=50e3, n_times=8263,
                   ha_range_h=4.0, freqs_hz=_chan(120.0, 168.0, 32), n_src=200, flux="powerlaw",
                   lm_max=0.05, noise_sigma=0.1, weights="uniform", N=8192, Nw=32, support=7,
                   sigma=1.0, dtype="c64", fov=0.2),
    # BASELINE.json configs[4]
    "hotspot": Config(name="hotspot", M=1_000_000_000, n_ant_core=42, n_ant_outer=20,
                      core_sigma_m=300.0, core_up_sigma_m=0.0, outer_rmin_m=1e3,
                      outer_rmax_m=50e3, n_times=66110, ha_range_h=4.0,
                      freqs_hz=_chan(120.0, 168.0, 8), n_src=50, flux="powerlaw", lm_max=0.15,
                      noise_sigma=0.01, weights="uniform", hotspot_frac=0.7,
                      hotspot_radius_lambda=200.0, hotspot_w_lambda=100.0, N=16384, Nw=16,
                      support=9, sigma=1.3, dtype="c64", fov=0.6),
}


def scaled(cfg: Config, M: int, **plan) -> Config:
    """Same recipe with fewer visibilities (and optionally another plan) -- the parity-test sizes."""
    return replace(cfg, M=int(M), **plan)


# ----------------------------------------------------------------------------------------------
# array, sources
# ----------------------------------------------------------------------------------------------

def antenna_enu(cfg: Config) -> torch.Tensor:
    """[n_ant, 3] float64 East, North, Up in metres (CPU)."""
    nc, no = cfg.n_ant_core, cfg.n_ant_outer
    i = torch.arange(nc + no, dtype=torch.int64)
    e = rng_normal(cfg.seed, _STREAM_ANT, i * 8 + 0) * cfg.core_sigma_m
    n = rng_normal(cfg.seed, _STREAM_ANT, i * 8 + 1) * cfg.core_sigma_m
    up = rng_normal(cfg.seed, _STREAM_ANT, i * 8 + 2) * cfg.core_up_sigma_m
    if no > 0:
        ur = rng_uniform(cfg.seed, _STREAM_ANT, i * 8 + 3)
        ua = rng_uniform(cfg.seed, _STREAM_ANT, i * 8 + 4)
        r = cfg.outer_rmin_m * torch.pow(torch.tensor(cfg.outer_rmax_m / cfg.outer_rmin_m,
                                                      dtype=torch.float64), ur)
        az = 2.0 * math.pi * ua
        outer = i >= nc
        e = torch.where(outer, r * torch.sin(az), e)
        n = torch.where(outer, r * torch.cos(az), n)
        up = torch.where(outer, torch.zeros_like(up), up)
    return torch.stack([e, n, up], dim=1)


def baselines_xyz(cfg: Config) -> torch.Tensor:
    """[n_bl, 3] float64 equatorial baseline vectors (Lx, Ly, Lz) in metres (CPU)."""
    enu = antenna_enu(cfg)
    phi = math.radians(cfg.lat_deg)
    e, n, up = enu[:, 0], enu[:, 1], enu[:, 2]
    x = -n * math.sin(phi) + up * math.cos(phi)
    y = e
    z = n * math.cos(phi) + up * math.sin(phi)
    xyz = torch.stack([x, y, z], dim=1)
    na = xyz.shape[0]
    ia, ib = torch.triu_indices(na, na, offset=1)
    return xyz[ib] - xyz[ia]


def sources(cfg: Config) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """(A, l, m) float64 tensors of length n_src (CPU)."""
    i = torch.arange(cfg.n_src, dtype=torch.int64)
    ua = rng_uniform(cfg.seed, _STREAM_SRC, i * 4 + 0)
    ul = rng_uniform(cfg.seed, _STREAM_SRC, i * 4 + 1)
    um = rng_uniform(cfg.seed, _STREAM_SRC, i * 4 + 2)
    if cfg.flux == "uniform":
        amp = 0.5 + 1.5 * ua
    elif cfg.flux == "powerlaw":
        amp = torch.clamp(0.05 * torch.pow(1.0 - ua, -1.0 / 1.5), max=10.0)
    else:
        raise ValueError(cfg.flux)
    l = (2.0 * ul - 1.0) * cfg.lm_max
    m = (2.0 * um - 1.0) * cfg.lm_max
    return amp, l, m


# ----------------------------------------------------------------------------------------------
# visibilities
# ----------------------------------------------------------------------------------------------

@dataclass
class Visibilities:
    u: torch.Tensor        # float32 [M] wavelengths
    v: torch.Tensor        # float32 [M]
    w: torch.Tensor        # float32 [M]
    vis: torch.Tensor      # complex64 [M]
    weight: torch.Tensor   # float32 [M]

    @property
    def M(self) -> int:
        return int(self.u.shape[0])

    def to(self, device) -> "Visibilities":
        return Visibilities(*(t.to(device) for t in (self.u, self.v, self.w, self.vis, self.weight)))

    def numpy(self):
        return tuple(t.detach().cpu().numpy() for t in (self.u, self.v, self.w, self.vis, self.weight))


def _uvw_rows(cfg: Config, rows: torch.Tensor, bl: torch.Tensor, freqs: torch.Tensor) -> Tuple[torch.Tensor, ...]:
    """float64 (u, v, w) in wavelengths for global row indices `rows` (int64, on the target device)."""
    n_bl, n_ch = cfg.n_bl, cfg.n_ch
    c = rows % n_ch
    tb = rows // n_ch
    b = tb % n_bl
    t = tb // n_bl
    ha_max = cfg.ha_range_h * (math.pi / 12.0)
    if cfg.n_times > 1:
        H = -ha_max + (2.0 * ha_max / (cfg.n_times - 1)) * t.to(torch.float64)
    else:
        H = torch.zeros_like(t, dtype=torch.float64)
    L = bl[b]
    Lx, Ly, Lz = L[:, 0], L[:, 1], L[:, 2]
    sd, cd = math.sin(math.radians(cfg.dec_deg)), math.cos(math.radians(cfg.dec_deg))
    sH, cH = torch.sin(H), torch.cos(H)
    inv_lambda = freqs[c] / C_LIGHT
    u = (sH * Lx + cH * Ly) * inv_lambda
    v = (-sd * cH * Lx + sd * sH * Ly + cd * Lz) * inv_lambda
    w = (cd * cH * Lx - cd * sH * Ly + sd * Lz) * inv_lambda
    return u, v, w


def generate(cfg: Config, device="cpu", chunk: int = 1 << 22, with_noise: bool = True) -> Visibilities:
    """Generate the whole configuration on `device` (chunked; float64 model phases on the
    fp32-rounded uvw, as the imaging side will see them)."""
    dev = torch.device(device)
    M = cfg.M
    if M > cfg.n_times * cfg.n_bl * cfg.n_ch:
        raise ValueError("config has fewer rows than M")
    bl = baselines_xyz(cfg).to(dev)
    freqs = torch.tensor(cfg.freqs_hz, dtype=torch.float64, device=dev)
    amp, sl, sm = sources(cfg)
    snm1 = -(sl * sl + sm * sm) / (1.0 + torch.sqrt(1.0 - sl * sl - sm * sm))
    amp_l, sl_l, sm_l, snm1_l = amp.tolist(), sl.tolist(), sm.tolist(), snm1.tolist()

    u_out = torch.empty(M, dtype=torch.float32, device=dev)
    v_out = torch.empty(M, dtype=torch.float32, device=dev)
    w_out = torch.empty(M, dtype=torch.float32, device=dev)
    vis_out = torch.empty(M, dtype=torch.complex64, device=dev)
    wt_out = torch.empty(M, dtype=torch.float32, device=dev)

    for start in range(0, M, chunk):
        stop = min(M, start + chunk)
        rows = torch.arange(start, stop, dtype=torch.int64, device=dev)
        u, v, w = _uvw_rows(cfg, rows, bl, freqs)
        if cfg.hotspot_frac > 0.0:
            sel = rng_uniform(cfg.seed, _STREAM_HOT, rows * 4 + 0) < cfg.hotspot_frac
            rr = cfg.hotspot_radius_lambda * torch.sqrt(rng_uniform(cfg.seed, _STREAM_HOT, rows * 4 + 1))
            th = 2.0 * math.pi * rng_uniform(cfg.seed, _STREAM_HOT, rows * 4 + 2)
            ww = cfg.hotspot_w_lambda * (2.0 * rng_uniform(cfg.seed, _STREAM_HOT, rows * 4 + 3) - 1.0)
            u = torch.where(sel, rr * torch.cos(th), u)
            v = torch.where(sel, rr * torch.sin(th), v)
            w = torch.where(sel, ww, w)
        u32, v32, w32 = u.to(torch.float32), v.to(torch.float32), w.to(torch.float32)
        ud, vd, wd = u32.to(torch.float64), v32.to(torch.float64), w32.to(torch.float64)
        re = torch.zeros(stop - start, dtype=torch.float64, device=dev)
        im = torch.zeros_like(re)
        for a, l, m, nm1 in zip(amp_l, sl_l, sm_l, snm1_l):
            # PAPER.md Eq. 1 (line 48) with I/n -> A: V = sum_s A_s exp(-2 pi i (u l + v m + w (n - 1)))
            ph = ud * l + vd * m + wd * nm1
            ph = (ph - torch.floor(ph)) * (2.0 * math.pi)
            re += a * torch.cos(ph)
            im -= a * torch.sin(ph)
        if with_noise and cfg.noise_sigma > 0.0:
            re += cfg.noise_sigma * rng_normal(cfg.seed, _STREAM_NOISE, rows * 2 + 0)
            im += cfg.noise_sigma * rng_normal(cfg.seed, _STREAM_NOISE, rows * 2 + 1)
        if cfg.weights == "unit":
            wt = torch.ones(stop - start, dtype=torch.float32, device=dev)
        else:
            wt = (0.5 + 0.5 * rng_uniform(cfg.seed, _STREAM_WEIGHT, rows)).to(torch.float32)
        u_out[start:stop] = u32
        v_out[start:stop] = v32
        w_out[start:stop] = w32
        vis_out[start:stop] = torch.complex(re.to(torch.float32), im.to(torch.float32))
        wt_out[start:stop] = wt
    return Visibilities(u_out, v_out, w_out, vis_out, wt_out)


def w_range(cfg: Config, vis: Visibilities) -> Tuple[float, float]:
    """(w_min, w_max) handed to the plan: the w extent of the visibilities whose (u, v) lie inside
    the mesh less a margin of support/2 + 1 cells (so no planes are spent on baselines that fall
    off the mesh anyway).  A data-side choice: any pair with w_max > w_min is a valid plan input."""
    du = 1.0 / cfg.fov
    lim = (cfg.N / 2 - (cfg.support + 1) / 2 - 1) * du
    inside = (vis.u.abs() < lim) & (vis.v.abs() < lim)
    if not bool(inside.any()):
        return -1.0, 1.0
    ws = vis.w[inside].to(torch.float64)
    lo, hi = float(ws.min()), float(ws.max())
    if not hi > lo:
        lo, hi = lo - 1.0, hi + 1.0
    return lo, hi


def plan_args(cfg: Config, vis: Optional[Visibilities] = None,
              w_min: Optional[float] = None, w_max: Optional[float] = None) -> dict:
    """Keyword arguments of rick_plan_create (include/rick_b200.h) for this configuration."""
    if w_min is None or w_max is None:
        w_min, w_max = w_range(cfg, vis)
    return dict(N=cfg.N, Nw=cfg.Nw, support=cfg.support, sigma=cfg.sigma,
                w_min=float(w_min), w_max=float(w_max), dl=cfg.dl)
