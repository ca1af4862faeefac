"""Seeded synthetic snapshot stacks shaped like the paper's workloads.

This module is shared by the CPU oracle's tests and by the CUDA path's tests and
bench.  It holds NONE of the method's arithmetic (no differences, ratios, tile
reductions, z-scores or DFTs): it only draws radio-sky-like fp32 images.

Stand-ins for the paper's MeerKAT / SKA AA2 / 50K x 50K workloads (the real
Measurement Set and the OSKAR/WSClean simulations are not available); the paper
itself times on pure Gaussian noise because run time is content independent
(section 3.2).  Recipe: SURVEY.md section 8(d), restated in DESIGN.md.

    x_s = steady + background + sum_j transient_j * active_j(s) + noise_s

* noise_s: i.i.d. N(0,1) fp32, independent per snapshot (and per channel)
* steady/background: identical in every snapshot
* PSF: circular Gaussian, sigma = FWHM / 2.35482, stamped within radius 6*FWHM;
  optional +-5 % ring sidelobes (config 2)
* fluxes are peak amplitudes in units of the noise sigma

Source parameters are always drawn on the CPU from `torch.Generator(seed)`, so a
stack has the same sources on every device.  The noise is drawn on the target
device; CPU and CUDA noise bits differ, which is harmless: a test always hands the
SAME buffer to both the oracle and the library.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional, Sequence, Tuple

import torch

BASE_SEED = 2509217540  # + cfg index (1..5); fits uint32


@dataclasses.dataclass(frozen=True)
class Transient:
    x: int
    y: int
    peak: float
    active: Tuple[int, ...]  # snapshot indices (0-based) in which it is on


@dataclasses.dataclass(frozen=True)
class StackConfig:
    name: str
    cfg_index: int
    L: int
    H: int
    W: int
    n_sources: int
    flux_lo: float
    flux_hi: float
    flux_dist: str = "loguniform"  # or "uniform"
    fwhm: float = 2.0
    sidelobes: bool = False
    n_background: int = 0
    n_transients: int = 0
    transient_mode: str = "none"  # fixed | periodic | near_bright | single
    transient_peak: float = 0.0
    tile: int = 32
    tau: float = 5.0
    n_channels: int = 1
    border: int = 16
    period: int = 8  # periodic transients: on when s % period == 3 % period

    def replace(self, **kw) -> "StackConfig":
        return dataclasses.replace(self, **kw)

    @property
    def seed(self) -> int:
        return BASE_SEED + self.cfg_index

    @property
    def n_pixels(self) -> int:
        return self.L * self.H * self.W


# BASELINE.json configs[0..4]
CONFIGS: Dict[str, StackConfig] = {
    "tiny": StackConfig("tiny", 1, L=8, H=256, W=256, n_sources=5, flux_lo=20.0, flux_hi=50.0,
                        flux_dist="uniform", fwhm=2.0, n_transients=1, transient_mode="fixed",
                        transient_peak=8.0, tau=6.0),
    "meerkat": StackConfig("meerkat", 2, L=64, H=2048, W=2048, n_sources=200, flux_lo=5.0, flux_hi=500.0,
                           fwhm=3.0, sidelobes=True, n_background=3, n_transients=1,
                           transient_mode="periodic", transient_peak=6.0, tau=5.0),
    "ska_aa2": StackConfig("ska_aa2", 3, L=32, H=8192, W=8192, n_sources=5000, flux_lo=5.0, flux_hi=1000.0,
                           fwhm=2.0, n_transients=20, transient_mode="near_bright", tau=5.0),
    "stream50k": StackConfig("stream50k", 4, L=4, H=50000, W=50000, n_sources=100000, flux_lo=5.0,
                             flux_hi=500.0, fwhm=2.0, n_transients=50, transient_mode="single",
                             transient_peak=7.0, tau=6.0),
    "imgfreq": StackConfig("imgfreq", 5, L=32, H=4096, W=4096, n_sources=1000, flux_lo=5.0, flux_hi=500.0,
                           fwhm=2.0, n_transients=5, transient_mode="periodic", transient_peak=5.0,
                           tau=6.0, n_channels=16),
    # NOT a BASELINE.json config: the shape of the paper's real-data run (1500 snapshots of 2 s,
    # 4096 x 4096, a 76 s pulsar = one pulse every 38 snapshots), used for a context line in DESIGN.md
    "psr_like": StackConfig("psr_like", 6, L=1500, H=4096, W=4096, n_sources=1000, flux_lo=5.0, flux_hi=500.0,
                            fwhm=2.0, n_transients=1, transient_mode="periodic", transient_peak=4.0,
                            tau=6.0, period=38),
}


def scaled(cfg: StackConfig, H: int, W: int, L: Optional[int] = None, name: Optional[str] = None) -> StackConfig:
    """Same recipe on a smaller image: source and transient counts scale with the area (at least 1)."""
    f = (H * W) / float(cfg.H * cfg.W)
    return cfg.replace(
        name=name or f"{cfg.name}_{H}x{W}", H=H, W=W, L=L or cfg.L,
        n_sources=max(1, int(round(cfg.n_sources * f))),
        n_transients=max(1, int(round(cfg.n_transients * f))) if cfg.n_transients else 0,
    )


def _loguniform(gen: torch.Generator, n: int, lo: float, hi: float) -> torch.Tensor:
    u = torch.rand(n, generator=gen, dtype=torch.float64)
    return torch.exp(math.log(lo) + u * (math.log(hi) - math.log(lo)))


def _uniform(gen: torch.Generator, n: int, lo: float, hi: float) -> torch.Tensor:
    return lo + (hi - lo) * torch.rand(n, generator=gen, dtype=torch.float64)


def _randint(gen: torch.Generator, n: int, lo: int, hi: int) -> torch.Tensor:
    """Integers uniform in [lo, hi)."""
    return torch.randint(lo, hi, (n,), generator=gen, dtype=torch.int64)


def _stamp(img: torch.Tensor, xs: torch.Tensor, ys: torch.Tensor, peaks: torch.Tensor, fwhm,
           sidelobes: bool, chunk: int = 8192) -> None:
    """Add one PSF per (x, y, peak) to img[H, W] in place.  `fwhm` is a float or a per-source tensor."""
    H, W = img.shape
    dev = img.device
    n = xs.numel()
    if n == 0:
        return
    fwhm_t = torch.as_tensor(fwhm, dtype=torch.float64).expand(n) if not torch.is_tensor(fwhm) else fwhm.double()
    fmax = float(fwhm_t.max())
    rad = int(math.ceil(6.0 * fmax))
    d = torch.arange(-rad, rad + 1, device=dev)
    dy, dx = torch.meshgrid(d, d, indexing="ij")
    r2 = (dx * dx + dy * dy).to(torch.float64).reshape(1, -1)
    r = torch.sqrt(r2)
    dxf, dyf = dx.reshape(1, -1), dy.reshape(1, -1)
    flat = img.view(-1)
    for i0 in range(0, n, chunk):
        sl = slice(i0, min(n, i0 + chunk))
        fw = fwhm_t[sl].to(dev).reshape(-1, 1)
        sig = fw / 2.35482
        prof = torch.exp(-0.5 * r2 / (sig * sig))
        prof = torch.where(r <= 6.0 * fw, prof, torch.zeros_like(prof))
        if sidelobes:
            ring_sig = fw / 2.355
            prof = prof - 0.05 * torch.exp(-0.5 * ((r - 1.5 * fw) / ring_sig) ** 2)
            prof = prof + 0.05 * torch.exp(-0.5 * ((r - 2.5 * fw) / ring_sig) ** 2)
        vals = (peaks[sl].to(dev).reshape(-1, 1) * prof).to(torch.float32)
        px = xs[sl].to(dev).reshape(-1, 1) + dxf
        py = ys[sl].to(dev).reshape(-1, 1) + dyf
        ok = (px >= 0) & (px < W) & (py >= 0) & (py < H)
        idx = (py * W + px)[ok]
        flat.index_put_((idx,), vals[ok], accumulate=True)


@dataclasses.dataclass
class Truth:
    cfg: StackConfig
    channel: int
    source_x: torch.Tensor
    source_y: torch.Tensor
    source_flux: torch.Tensor
    transients: List[Transient]


def draw_truth(cfg: StackConfig, channel: int = 0) -> Truth:
    """Source and transient parameters (device independent, CPU generator)."""
    gen = torch.Generator(device="cpu")
    gen.manual_seed(cfg.seed)
    b = min(cfg.border, max(0, min(cfg.H, cfg.W) // 2 - 1))
    n = cfg.n_sources
    sx = _randint(gen, n, b, max(b + 1, cfg.W - b))
    sy = _randint(gen, n, b, max(b + 1, cfg.H - b))
    if cfg.flux_dist == "uniform":
        flux = _uniform(gen, n, cfg.flux_lo, cfg.flux_hi)
    else:
        flux = _loguniform(gen, n, cfg.flux_lo, cfg.flux_hi)
    alpha = _uniform(gen, n, -1.5, 0.5)  # spectral index, used by the multi-channel config only
    tr: List[Transient] = []
    m = cfg.n_transients
    if cfg.transient_mode == "fixed":
        # BASELINE.json configs[0]: fixed pixel, on in snapshots 2 and 6
        fx = min(77, cfg.W - 1 - b) if cfg.W > 77 + b else cfg.W // 3
        fy = min(100, cfg.H - 1 - b) if cfg.H > 100 + b else cfg.H // 3
        tr.append(Transient(int(fx), int(fy), cfg.transient_peak, tuple(s for s in (2, 6) if s < cfg.L)))
    elif cfg.transient_mode == "periodic":
        tx = _randint(gen, m, b, max(b + 1, cfg.W - b))
        ty = _randint(gen, m, b, max(b + 1, cfg.H - b))
        act = tuple(s for s in range(cfg.L) if s % cfg.period == 3 % cfg.period)
        for j in range(m):
            tr.append(Transient(int(tx[j]), int(ty[j]), cfg.transient_peak, act))
    elif cfg.transient_mode == "near_bright":
        bright = torch.nonzero(flux >= 100.0).flatten()
        if bright.numel() == 0:
            bright = torch.argsort(flux, descending=True)[: max(1, m)]
        pick = bright[torch.randperm(bright.numel(), generator=gen)[:m]]
        dist = _uniform(gen, pick.numel(), 4.0, 8.0)
        ang = _uniform(gen, pick.numel(), 0.0, 2.0 * math.pi)
        n_on = max(1, int(round(0.1 * cfg.L)))
        for j, h in enumerate(pick.tolist()):
            x = int(round(float(sx[h]) + float(dist[j]) * math.cos(float(ang[j]))))
            y = int(round(float(sy[h]) + float(dist[j]) * math.sin(float(ang[j]))))
            x = min(max(x, 0), cfg.W - 1)
            y = min(max(y, 0), cfg.H - 1)
            on = torch.randperm(cfg.L, generator=gen)[:n_on].sort().values
            tr.append(Transient(x, y, float(flux[h]) / 20.0, tuple(int(v) for v in on)))
    elif cfg.transient_mode == "single":
        tx = _randint(gen, m, b, max(b + 1, cfg.W - b))
        ty = _randint(gen, m, b, max(b + 1, cfg.H - b))
        ts = _randint(gen, m, 0, cfg.L)
        for j in range(m):
            tr.append(Transient(int(tx[j]), int(ty[j]), cfg.transient_peak, (int(ts[j]),)))
    if cfg.n_channels > 1:
        nu = 1.0 + channel / float(cfg.n_channels - 1)
        flux = flux * torch.pow(torch.tensor(nu, dtype=torch.float64), alpha)
        tr = [Transient(t.x, t.y, t.peak * nu ** -3.0, t.active) for t in tr]
    return Truth(cfg, channel, sx, sy, flux, tr)


def channel_fwhm(cfg: StackConfig, channel: int) -> float:
    if cfg.n_channels > 1:
        return cfg.fwhm / (1.0 + channel / float(cfg.n_channels - 1))
    return cfg.fwhm


def steady_image(cfg: StackConfig, truth: Truth, device="cpu") -> torch.Tensor:
    """steady sources + smooth background, [H, W] fp32 on `device`."""
    img = torch.zeros((cfg.H, cfg.W), dtype=torch.float32, device=device)
    fw = channel_fwhm(cfg, truth.channel)
    _stamp(img, truth.source_x, truth.source_y, truth.source_flux, fw, cfg.sidelobes)
    if cfg.n_background:
        gen = torch.Generator(device="cpu")
        gen.manual_seed(cfg.seed + 7919)
        cx = _uniform(gen, cfg.n_background, 0.0, cfg.W)
        cy = _uniform(gen, cfg.n_background, 0.0, cfg.H)
        sg = _uniform(gen, cfg.n_background, cfg.H / 4.0, cfg.H / 2.0)
        yy = torch.arange(cfg.H, device=device, dtype=torch.float32).reshape(-1, 1)
        xx = torch.arange(cfg.W, device=device, dtype=torch.float32).reshape(1, -1)
        for k in range(cfg.n_background):
            img += 2.0 * torch.exp(-0.5 * (((xx - float(cx[k])) / float(sg[k])) ** 2
                                            + ((yy - float(cy[k])) / float(sg[k])) ** 2))
    return img


def snapshot(cfg: StackConfig, truth: Truth, steady: torch.Tensor, s: int,
             out: Optional[torch.Tensor] = None, noise_sigma: float = 1.0) -> torch.Tensor:
    """Snapshot s ([H, W] fp32) on steady.device; written into `out` when given."""
    dev = steady.device
    gen = torch.Generator(device=dev)
    gen.manual_seed((cfg.seed * 1000003 + truth.channel * 4099 + s) % (2 ** 63 - 1))
    if out is None:
        out = torch.empty_like(steady)
    if noise_sigma > 0.0:
        out.normal_(0.0, noise_sigma, generator=gen)
        out += steady
    else:
        out.copy_(steady)
    on = [t for t in truth.transients if s in t.active]
    if on:
        fw = channel_fwhm(cfg, truth.channel)
        _stamp(out,
               torch.tensor([t.x for t in on], dtype=torch.int64),
               torch.tensor([t.y for t in on], dtype=torch.int64),
               torch.tensor([t.peak for t in on], dtype=torch.float64), fw, False)
    return out


def make_stack(cfg: StackConfig, device="cpu", channel: int = 0, noise_sigma: float = 1.0,
               out: Optional[torch.Tensor] = None) -> Tuple[torch.Tensor, Truth]:
    """The whole [L, H, W] fp32 stack on `device` plus the truth record."""
    truth = draw_truth(cfg, channel)
    steady = steady_image(cfg, truth, device)
    if out is None:
        out = torch.empty((cfg.L, cfg.H, cfg.W), dtype=torch.float32, device=device)
    for s in range(cfg.L):
        snapshot(cfg, truth, steady, s, out=out[s], noise_sigma=noise_sigma)
    return out, truth


def gaussian_noise_stack(L: int, H: int, W: int, seed: int = BASE_SEED, device="cpu") -> torch.Tensor:
    """Pure N(0,1) snapshots: the paper's own timing input."""
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    return torch.randn((L, H, W), dtype=torch.float32, device=device, generator=gen)
