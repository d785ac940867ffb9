"""Detector-count model and the five workload recipes of BASELINE.json (C1..C5).

counts = noise(flat * exp(-p)) + dark, rounded and clipped to uint16, where p are
the closed-form line integrals of the phantom.  Every random draw is seeded per
slice row, so any subset of rows can be generated independently and reproducibly.
No reconstruction arithmetic lives here.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from .phantom import Ellipsoids, head_phantom, line_integrals, random_ellipsoids

BASE_SEED = 20220908


@dataclass
class Workload:
    name: str
    n: int                 # detector width = image side
    nproj: int
    nz_total: int          # slices (detector rows) in the whole volume
    nz_chunk: int
    center: float
    dtype: str             # "f32" | "f16" | "f16_out32"
    filter: str            # "ramp" | "shepp" | "parzen"
    flat_level: float
    dark_level: float
    noise: str             # "poisson" | "gauss0.5%" | "none"
    nframes: int           # flat/dark frames to average
    seed: int
    phantom: Ellipsoids = field(repr=False, default=None)

    @property
    def theta(self) -> np.ndarray:
        return make_theta(self.nproj)


def make_theta(nproj: int) -> np.ndarray:
    """nproj angles equally spaced over [0, pi), float32 radians."""
    return (np.arange(nproj, dtype=np.float64) * (np.pi / nproj)).astype(np.float32)


def _rescale_to_p999(ph: Ellipsoids, n, nproj, center, nz_total, target=3.0) -> Ellipsoids:
    """Scale all mu so the 99.9th-percentile line integral (estimated on 16 angles x
    16 rows) equals `target` (5 % transmission): keeps the detector from starving
    when hundreds of ellipsoids overlap."""
    th = make_theta(nproj)[:: max(1, nproj // 16)][:16]
    rows = np.linspace(0, nz_total - 1, 16).round().astype(int)
    p = line_integrals(ph, th, n, center, rows, nz_total)
    q = float(np.quantile(p, 0.999))
    return ph.scaled(target / q) if q > 0 else ph


CONFIGS = ("C1", "C2", "C3", "C4", "C5")


def make_workload(name: str, scale: int = 1, dtype: str | None = None) -> Workload:
    """Recipe `name` in C1..C5.  `scale` > 1 divides every size by `scale` (same
    phantom in relative units) for down-sized parity runs of the large configs."""
    idx = CONFIGS.index(name)
    seed = BASE_SEED + idx
    if name == "C1":
        n, nproj, nzt, nzc, c = 128, 180, 8, 8, 64.0
        w = Workload(name, n, nproj, nzt, nzc, c, "f32", "shepp", 30000.0, 100.0, "poisson", 1, seed)
        n, nproj, nzt = n // scale, nproj // scale, max(2, nzt // scale)
        w.n, w.nproj, w.nz_total, w.nz_chunk, w.center = n, nproj, nzt, min(nzc, nzt), c / scale
        w.phantom = head_phantom(n, nzt, 0.02)
        return w
    spec = {
        # n, nproj, nz_total, chunk, centre offset from n/2, count, axes, dtype, flat, noise, frames
        "C2": (512, 720, 512, 32, 0.0, 40, (0.02, 0.12), "f32", 30000.0, "poisson", 1),
        "C3": (1024, 1500, 1024, 16, 3.5, 200, (0.01, 0.08), "f16", 30000.0, "gauss0.5%", 1),
        "C4": (2048, 2048, 2048, 32, 0.0, 500, (0.005, 0.06), "f16", 3500.0, "poisson", 10),
        "C5": (4096, 4000, 256, 32, 17.5, 300, (0.005, 0.06), "f16_out32", 3500.0, "poisson", 10),
    }[name]
    n, nproj, nzt, nzc, coff, cnt, axes, dt, flat, noise, frames = spec
    n, nproj, nzt = n // scale, max(8, nproj // scale), max(2, nzt // scale)
    c = n / 2.0 + coff   # the (half-pixel) offset is kept as is when down-scaling
    w = Workload(name, n, nproj, nzt, min(nzc, nzt), c, dtype or dt, "parzen", flat, 100.0, noise,
                 frames, seed)
    ph = random_ellipsoids(cnt, n, nzt, seed, axes_frac=axes)
    if name != "C2":
        ph = _rescale_to_p999(ph, n, nproj, c, nzt)
    w.phantom = ph
    return w


def make_flat_dark(w: Workload, z_rows):
    """Per-row flat gain and dark offset, plus the averaged float32 flat/dark the
    reconstruction receives.  Returns (flat_f32[r][n], dark_f32[r][n], flat_frames_u16
    [K][r][n], dark_frames_u16[K][r][n]); the float fields are the float32 mean of
    the K uint16 frames (sum is exact in fp32, one division)."""
    z_rows = np.asarray(z_rows)
    K = w.nframes
    ff = np.empty((K, len(z_rows), w.n), dtype=np.uint16)
    df = np.empty((K, len(z_rows), w.n), dtype=np.uint16)
    for r, iz in enumerate(z_rows):
        rng = np.random.default_rng([w.seed, 7, int(iz)])
        gain = w.flat_level * (1.0 + 0.02 * rng.standard_normal(w.n))
        doff = w.dark_level + 3.0 * rng.standard_normal(w.n)
        for k in range(K):
            if K == 1:
                fk, dk = gain + doff, doff
            else:
                fk = rng.poisson(np.clip(gain, 0, None)) + doff + 1.5 * rng.standard_normal(w.n)
                dk = doff + 1.5 * rng.standard_normal(w.n)
            ff[k, r] = np.clip(np.rint(fk), 0, 65535).astype(np.uint16)
            df[k, r] = np.clip(np.rint(dk), 0, 65535).astype(np.uint16)
    flat = (ff.astype(np.float32).sum(axis=0, dtype=np.float32) / np.float32(K)).astype(np.float32)
    dark = (df.astype(np.float32).sum(axis=0, dtype=np.float32) / np.float32(K)).astype(np.float32)
    return flat, dark, ff, df


def make_counts(w: Workload, z_rows, noise: bool = True):
    """uint16 projections raw[nproj][r][n] for the slice rows z_rows, with the flat
    gain / dark offset of those rows.  Returns (raw_u16, p_float64) where p are the
    noise-free line integrals (ground truth for pins)."""
    z_rows = np.asarray(z_rows)
    p = line_integrals(w.phantom, w.theta, w.n, w.center, z_rows, w.nz_total)
    raw = np.empty((w.nproj, len(z_rows), w.n), dtype=np.uint16)
    for r, iz in enumerate(z_rows):
        rng = np.random.default_rng([w.seed, 7, int(iz)])     # same stream head as make_flat_dark
        gain = w.flat_level * (1.0 + 0.02 * rng.standard_normal(w.n))
        doff = w.dark_level + 3.0 * rng.standard_normal(w.n)
        rng = np.random.default_rng([w.seed, 11, int(iz)])
        sig = np.clip(gain, 0, None)[None, :] * np.exp(-p[:, r, :])
        if not noise or w.noise == "none":
            cnt = sig
        elif w.noise == "poisson":
            cnt = rng.poisson(sig).astype(np.float64)
        else:  # 0.5 % multiplicative Gaussian detector noise
            cnt = sig * (1.0 + 0.005 * rng.standard_normal(sig.shape))
        raw[:, r, :] = np.clip(np.rint(cnt + doff[None, :]), 0, 65535).astype(np.uint16)
    return raw, p


def make_counts_torch(w: Workload, z_rows, device="cuda"):
    """The same recipe as make_counts/make_flat_dark evaluated with torch on `device`, for the
    large configs (C3..C5) where numpy would take minutes.  Random draws come from a torch
    generator seeded with (w.seed, first row), so they differ from the numpy path; the SAME
    arrays are given to the CUDA path and (copied to the host) to the oracle.
    Returns (raw_u16[nproj][r][n], flat_frames_u16[K][r][n], dark_frames_u16[K][r][n]) on device."""
    import torch

    z_rows = np.asarray(z_rows)
    g = torch.Generator(device=device)
    g.manual_seed(int(w.seed) * 100003 + int(z_rows[0]))
    p = line_integrals(w.phantom, w.theta, w.n, w.center, z_rows, w.nz_total, xp=torch,
                       dtype=torch.float32, device=device)
    R, n, K = len(z_rows), w.n, w.nframes
    gain = w.flat_level * (1.0 + 0.02 * torch.randn((R, n), generator=g, device=device))
    doff = w.dark_level + 3.0 * torch.randn((R, n), generator=g, device=device)
    sig = gain.clamp_min(0)[None] * torch.exp(-p)
    if w.noise == "poisson":
        cnt = torch.poisson(sig, generator=g)
    elif w.noise == "none":
        cnt = sig
    else:
        cnt = sig * (1.0 + 0.005 * torch.randn(sig.shape, generator=g, device=device))
    raw = (cnt + doff[None]).round().clamp(0, 65535).to(torch.int32).to(torch.uint16)
    if K == 1:
        ff, df = (gain + doff)[None], doff[None]
    else:
        ff = torch.poisson(gain.clamp_min(0)[None].expand(K, R, n), generator=g) + doff[None] \
            + 1.5 * torch.randn((K, R, n), generator=g, device=device)
        df = doff[None] + 1.5 * torch.randn((K, R, n), generator=g, device=device)
    ff = ff.round().clamp(0, 65535).to(torch.int32).to(torch.uint16)
    df = df.round().clamp(0, 65535).to(torch.int32).to(torch.uint16)
    return raw, ff, df
