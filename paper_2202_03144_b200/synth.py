"""Seeded synthetic scans shaped like the paper's beamline workloads.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path: it draws
objects, probes, scan positions and photon counts.  It holds none of the reconstruction
arithmetic: it never forms an update, a projection or an error.  The one physical formula it
needs is the far-field measurement model  I_j = sum_k |FFT2(P_k * O[r_j])|^2  (BASELINE.json
configs[0], "Intensities: |FFT2(P*O_j)|^2"), evaluated in float64 with the *library* FFT
(scipy.fft / pocketfft), which neither the oracle (own radix-2 FFT) nor the CUDA kernels use.

Stand-in statement: the paper measures on APS beamline data (Eiger-500K crops, kHz fly scans,
PAPER.md:29) and on its own `-simulate=1` images; neither is available, so
these generators stand in for them.  The recipe (readings R10-R19 of SURVEY.md 8(c), table in
8(d)) is restated in DESIGN.md section 4.

Conventions: positions are int32 (y, x) top-left corners; intensities are in FFT order (DC at
[0, 0]); complex arrays are complex128 here and cast by the consumer.
"""
from __future__ import annotations

import dataclasses
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import scipy.fft
import scipy.ndimage

MASK_U16 = 65535  # uint16 sentinel "no constraint" (reading R3/R11)


@dataclasses.dataclass
class Scan:
    name: str
    algorithm: str            # "DM" | "EPIE_MB" | "LSQML"
    n: int                    # frame side N
    obj_true: np.ndarray      # (H, W) complex128
    probe_true: np.ndarray    # (K, N, N) complex128, photon-scaled
    obj0: np.ndarray          # (H, W) complex128 initial guess (flat 1+0i)
    probe0: np.ndarray        # (K, N, N) complex128 initial guess (= probe_true, R19)
    pos: np.ndarray           # (J, 2) int32 (y, x)
    intensities: np.ndarray   # (J, N, N) float32 (negative = masked) or uint16 (65535 = masked)
    iterations: int
    params: dict              # batch_size, pbound, ... (defaults elsewhere)
    noise_floor: float        # mean (sqrt(n) - sqrt(lambda))^2 over unmasked pixels (R6)

    @property
    def n_pos(self) -> int:
        return int(self.pos.shape[0])

    @property
    def n_modes(self) -> int:
        return int(self.probe_true.shape[0])


# ----------------------------------------------------------------------------- objects (R14)
def make_object(h: int, w: int, seed: int) -> np.ndarray:
    """Amplitude: 5x5 periodic box filter of U(0,1), min-max -> [0.8, 1.0]; phase: periodic
    Gaussian filter (sigma 3 px) of N(0,1), min-max -> [-0.5, 0.5] rad.  Amplitude drawn first."""
    rng = np.random.default_rng(seed)
    a = rng.random((h, w))
    p = rng.standard_normal((h, w))
    a = scipy.ndimage.uniform_filter(a, size=5, mode="wrap")
    p = scipy.ndimage.gaussian_filter(p, sigma=3.0, mode="wrap")
    a = 0.8 + 0.2 * (a - a.min()) / (a.max() - a.min())
    p = -0.5 + (p - p.min()) / (p.max() - p.min())
    return a * np.exp(1j * p)


# ----------------------------------------------------------------------------- probes
def _radius_grid(n: int):
    y, x = np.mgrid[0:n, 0:n].astype(np.float64)
    y -= n // 2
    x -= n // 2
    return y, x, np.hypot(y, x)


def probe_disk(n: int, radius: float, chirp: float | None = None) -> np.ndarray:
    """R13: hard-edged Gaussian-apodised disk with quadratic phase."""
    _, _, r = _radius_grid(n)
    c = (4.0 / radius ** 2) if chirp is None else chirp
    return (r <= radius) * np.exp(-r ** 2 / (2 * radius ** 2)) * np.exp(1j * c * r ** 2)


def probe_zone(n: int, radius: float) -> np.ndarray:
    """R15: real-space chirped annulus (12 Fresnel zones, central stop R/4)."""
    _, _, r = _radius_grid(n)
    return ((r >= radius / 4) & (r <= radius)) * np.exp(-1j * np.pi * r ** 2 * 12.0 / radius ** 2)


def probe_modes(base: np.ndarray, fractions=(0.80, 0.15, 0.05)) -> np.ndarray:
    """R18: Gram-Schmidt of {P, x*P, y*P}; mode k carries fractions[k] of sum|P|^2."""
    n = base.shape[0]
    y, x, _ = _radius_grid(n)
    cand = [base, x * base, y * base][: len(fractions)]
    out = []
    for v in cand:
        v = v.astype(np.complex128).copy()
        for u in out:
            v -= u * (np.vdot(u, v) / np.vdot(u, u))
        out.append(v)
    total = float(np.sum(np.abs(base) ** 2))
    return np.stack([u * np.sqrt(f * total / float(np.sum(np.abs(u) ** 2)))
                     for u, f in zip(out, fractions)])


# ----------------------------------------------------------------------------- positions
def raster_positions(rows, cols, step, offset, jitter=0, seed=None, count=None) -> np.ndarray:
    yy, xx = np.mgrid[0:rows, 0:cols]
    pos = np.stack([yy.ravel() * step + offset[0], xx.ravel() * step + offset[1]], 1)
    if count is not None:
        pos = pos[:count]
    if jitter:
        rng = np.random.default_rng(seed)
        pos = pos + rng.integers(-jitter, jitter + 1, size=pos.shape)
    return pos.astype(np.int32)


def fermat_positions(j: int, h: int, n: int) -> np.ndarray:
    """R16: r = c*sqrt(k+1/2), theta = k*pi*(3-sqrt 5), scaled to fit the object."""
    k = np.arange(j, dtype=np.float64)
    half = (h - n) / 2.0
    c = (half - 2.0) / np.sqrt(j)
    r = c * np.sqrt(k + 0.5)
    th = k * np.pi * (3.0 - np.sqrt(5.0))
    pos = np.stack([half + r * np.sin(th), half + r * np.cos(th)], 1)
    return np.rint(pos).astype(np.int32)


# ----------------------------------------------------------------------------- measurement model
def _model_chunk(obj, probe, pos):
    n = probe.shape[-1]
    out = np.empty((len(pos), n, n), np.float64)
    for i, (y, x) in enumerate(pos):
        f = scipy.fft.fft2(probe * obj[None, y:y + n, x:x + n], axes=(-2, -1))
        out[i] = np.sum(f.real ** 2 + f.imag ** 2, axis=0)
    return out


def model_intensity(obj, probe, pos, threads: int = 8, chunk: int = 64):
    """Yield (start, lambda[start:start+len]) noiseless intensities in float64, chunk by chunk."""
    starts = list(range(0, len(pos), chunk))
    with ThreadPoolExecutor(threads) as ex:
        for s, lam in zip(starts, ex.map(lambda s: _model_chunk(obj, probe, pos[s:s + chunk]), starts)):
            yield s, lam


def simulate(obj, probe, pos, peak, poisson_seed, dtype, threads: int = 8):
    """R19: scale the probe so the brightest noiseless pixel equals `peak`, then draw Poisson
    counts (one child stream of `poisson_seed` per 64-frame chunk, so the result does not depend
    on the thread count).  `peak=None`: noiseless float32, no scaling (cfg0).  uint16: counts
    clipped to 65535 = mask sentinel (R11)."""
    j, n = len(pos), probe.shape[-1]
    if peak is None:
        out = np.empty((j, n, n), np.float32)
        for s, lam in model_intensity(obj, probe, pos, threads):
            out[s:s + len(lam)] = lam
        return probe, out, 0.0
    mx = max(float(lam.max()) for _, lam in model_intensity(obj, probe, pos, threads))
    probe = probe * np.sqrt(peak / mx)
    out = np.empty((j, n, n), dtype)
    seeds = np.random.SeedSequence(poisson_seed).spawn((j + 63) // 64)

    def chunk(s):
        lam = _model_chunk(obj, probe, pos[s:s + 64])
        cnt = np.random.default_rng(seeds[s // 64]).poisson(lam)
        if dtype == np.uint16:
            cnt = np.minimum(cnt, MASK_U16)
            ok = cnt < MASK_U16
        else:
            ok = np.ones(cnt.shape, bool)
        out[s:s + len(lam)] = cnt
        return float(np.sum((np.sqrt(cnt[ok]) - np.sqrt(lam[ok])) ** 2)), int(ok.sum())

    with ThreadPoolExecutor(threads) as ex:
        parts = list(ex.map(chunk, range(0, j, 64)))
    nf_sum, nf_cnt = sum(p[0] for p in parts), sum(p[1] for p in parts)
    return probe, out, nf_sum / max(nf_cnt, 1)


# ----------------------------------------------------------------------------- the configs
def make_config(i: int, n_pos: int | None = None, threads: int = 8, scale: int = 1, replica: int = 0) -> Scan:
    """Config i of BASELINE.json / SURVEY.md 8(d).  `n_pos` truncates the scan (first n_pos
    positions of the same generator; used where the oracle cannot hold the full scan).
    `scale` > 1 divides N, H and the probe radius (same recipe, reduced size, for CPU tests).
    `replica` r > 0 shifts every seed by 10*r: an independent scan of the same shape (bench.py
    --gpus N runs one replica per GPU)."""
    so, sj, sp = 1000 + i + 10 * replica, 2000 + i + 10 * replica, 3000 + i + 10 * replica
    s = scale
    if i == 0:
        n, h, alg, its = 64 // s, 192 // s, "DM", 10
        base = probe_disk(n, 20 / s, 0.01 * s * s)[None]
        pos = raster_positions(8, 8, 16 // s, (8 // s, 8 // s))
        peak, dt, params = None, np.float32, dict(pbound=0.0)
    elif i == 1:
        n, h, alg, its = 128 // s, 1024 // s, "EPIE_MB", 50
        base = probe_disk(n, 40 / s)[None]
        pos = raster_positions(32, 32, 24 // s, (76 // s, 76 // s), jitter=2, seed=sj)
        peak, dt, params = 1e4, np.float32, dict(batch_size=256, pbound_dm=0.12)
    elif i == 2:
        n, h, alg, its = 256 // s, 4096 // s, "DM", 100
        base = probe_zone(n, 80 / s)[None]
        pos = fermat_positions(10000, h, n)
        peak, dt, params = 1e5, np.uint16, dict(pbound=0.5)
    elif i == 3:
        n, h, alg, its = 256 // s, 6144 // s, "LSQML", 50
        base = probe_modes(probe_disk(n, 80 / s))
        step = 40 // s
        off = ((h - n - 140 * step) // 2, (h - n - 141 * step) // 2)
        pos = raster_positions(141, 142, step, off, jitter=3 if s == 1 else 1, seed=sj, count=20000)
        peak, dt, params = 1e4, np.uint16, dict(batch_size=512)
    elif i == 4:
        n, h, alg, its = 512 // s, 8192 // s, "DM", 20
        base = probe_zone(n, 160 / s)[None]
        pos = fermat_positions(16384, h, n)
        peak, dt, params = 1e5, np.uint16, dict(pbound=0.5)
    else:
        raise ValueError(f"no config {i}")
    if n_pos is not None:
        pos = pos[:n_pos]
    assert pos.min() >= 0 and pos.max() + n <= h, "scan does not fit the object"
    obj = make_object(h, h, so)
    probe, inten, nf = simulate(obj, base, pos, peak, sp, dt, threads)
    return Scan(name=f"cfg{i}" + (f"/{s}" if s > 1 else ""), algorithm=alg, n=n, obj_true=obj,
                probe_true=probe, obj0=np.ones_like(obj), probe0=probe.copy(), pos=pos,
                intensities=inten, iterations=its, params=params, noise_floor=nf)


def make_custom(n, h, j_side, step, k=1, peak=None, seed=7, dtype=np.float32, jitter=0,
                probe_kind="disk", threads: int = 4) -> Scan:
    """Small raster scans of arbitrary shape for unit tests (same building blocks)."""
    radius = n * 0.3125
    base = probe_disk(n, radius) if probe_kind == "disk" else probe_zone(n, radius)
    base = probe_modes(base)[:k] if k > 1 else base[None]
    off = (h - n - (j_side - 1) * step) // 2
    pos = raster_positions(j_side, j_side, step, (off, off), jitter=jitter, seed=seed + 1)
    obj = make_object(h, h, seed)
    probe, inten, nf = simulate(obj, base, pos, peak, seed + 2, dtype, threads)
    return Scan(name=f"custom{n}", algorithm="DM", n=n, obj_true=obj, probe_true=probe,
                obj0=np.ones_like(obj), probe0=probe.copy(), pos=pos, intensities=inten,
                iterations=5, params={}, noise_floor=nf)
