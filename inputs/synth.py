"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic (no kernel, no correction, no
FFT, no gridding): it only draws images, (u, v) coordinates, weights and noise.
It is the one module shared by the CPU oracle's tests and the CUDA path, so that
both sides see the very same arrays (task rule 3: "only the seeded input
generators serve both, from a module of their own").

The paper's own benchmarks use synthetic data: "random Gaussian-density (u,v)"
scaled to +-pi per axis, Kaiser-Bessel J=4, so these generators
stand in for nothing external.  Coordinates are returned in *oversampled-grid
cells* (period K = 2n, DC at 0); u_cells = omega * K / (2 pi) for the paper's
radians-per-pixel omega.

Recipe per config: DESIGN.md "Input recipe"; SURVEY.md 8(d) "Synthetic inputs".
All draws go through numpy's PCG64 seeded with (1000 + config index, substream).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

# sub-stream ids
STREAM_IMAGE, STREAM_UV, STREAM_W, STREAM_NOISE, STREAM_TEST, STREAM_SHUFFLE = 1, 2, 3, 4, 5, 6


def rng_for(seed: int, stream: int) -> np.random.Generator:
    """Independent, reproducible generator for (seed, stream)."""
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([int(seed), int(stream)])))


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json config (index 1..5)."""
    index: int
    name: str
    n: int               # image side
    J: int               # kernel support (taps per axis)
    M: int               # number of visibilities
    dtype: str           # "c64" | "c128"
    uv: str              # "gauss" | "vla27" | "ska197"
    sigma_div: float     # gaussian sigma = K / sigma_div cells (gauss only)
    weights: str         # "unit" | "uniform"
    kernel_mode: str     # "analytic" | "table"
    table_R: int = 4096  # table samples per unit (table mode)

    @property
    def K(self) -> int:
        return 2 * self.n

    @property
    def seed(self) -> int:
        return 1000 + self.index


CONFIGS = {
    1: Config(1, "tiny", 128, 4, 10_000, "c128", "gauss", 8.0, "unit", "analytic"),
    2: Config(2, "small", 256, 4, 250_000, "c128", "gauss", 6.0, "uniform", "analytic"),
    3: Config(3, "vla27", 1024, 4, 10_000_000, "c64", "vla27", 0.0, "uniform", "analytic"),
    4: Config(4, "gauss1e8", 2048, 6, 100_000_000, "c64", "gauss", 6.0, "uniform", "analytic"),
    5: Config(5, "ska197", 4096, 4, 500_000_000, "c64", "ska197", 0.0, "uniform", "table", 4096),
}


def real_dtype(dtype: str):
    return np.float32 if dtype == "c64" else np.float64


def complex_dtype(dtype: str):
    return np.complex64 if dtype == "c64" else np.complex128


# --------------------------------------------------------------------------- images
def make_image(n: int, seed: int, dtype: str = "c128") -> np.ndarray:
    """n x n complex image: 20 point sources (amplitude U[0,1], random pixels, added)
    plus 3 Gaussian blobs of sigma 4 px (centres U[n/4, 3n/4)^2, peak U[0.5, 1],
    set exactly to zero beyond 6 sigma).  Imaginary part zero (the sky is real,
    PAPER.md:53) but the array is complex because the operator is complex->complex.
    BASELINE.json configs[0]; SURVEY.md 8(d) row 1."""
    rng = rng_for(seed, STREAM_IMAGE)
    img = np.zeros((n, n), dtype=np.float64)
    py = rng.integers(0, n, size=20)
    px = rng.integers(0, n, size=20)
    amp = rng.uniform(0.0, 1.0, size=20)
    for a, yy, xx in zip(amp, py, px):
        img[yy, xx] += a
    sigma = 4.0
    for _ in range(3):
        cy, cx = rng.uniform(n / 4, 3 * n / 4, size=2)
        peak = rng.uniform(0.5, 1.0)
        y0, y1 = max(0, int(cy - 6 * sigma)), min(n, int(cy + 6 * sigma) + 2)
        x0, x1 = max(0, int(cx - 6 * sigma)), min(n, int(cx + 6 * sigma) + 2)
        yy, xx = np.mgrid[y0:y1, x0:x1]
        r2 = (yy - cy) ** 2 + (xx - cx) ** 2
        blob = peak * np.exp(-r2 / (2 * sigma * sigma))
        blob[r2 > (6 * sigma) ** 2] = 0.0
        img[y0:y1, x0:x1] += blob
    return img.astype(complex_dtype(dtype))


def random_complex(shape, seed: int, stream: int = STREAM_TEST, dtype: str = "c128") -> np.ndarray:
    """i.i.d. complex standard normal (test vectors for the adjoint identity)."""
    rng = rng_for(seed, stream)
    rd = real_dtype(dtype)
    out = np.empty(shape, dtype=complex_dtype(dtype))
    out.real = rng.standard_normal(shape, dtype=rd)
    out.imag = rng.standard_normal(shape, dtype=rd)
    return out


# --------------------------------------------------------------------------- uv
def uv_gaussian(M: int, K: int, J: int, sigma_div: float, seed: int, dtype: str = "c128") -> np.ndarray:
    """[M][2] (u, v) in grid cells: i.i.d. N(0, (K/sigma_div)^2) per axis, rejection-
    truncated to |u|, |v| < K/2 - J (BASELINE.json configs[0,1,3]; PAPER.md:534 uses a
    Gaussian density scaled to +-pi).  Stored in the config's real dtype."""
    rng = rng_for(seed, STREAM_UV)
    rd = real_dtype(dtype)
    lim = K / 2 - J
    sigma = K / sigma_div
    out = np.empty((M, 2), dtype=rd)
    filled = 0
    chunk = 1 << 22
    while filled < M:
        want = min(chunk, int((M - filled) * 1.05) + 1024)
        c = rng.standard_normal((want, 2)) * sigma
        c = c.astype(rd)                       # truncate AFTER rounding to storage
        ok = (np.abs(c[:, 0]) < lim) & (np.abs(c[:, 1]) < lim)
        c = c[ok]
        take = min(len(c), M - filled)
        out[filled:filled + take] = c[:take]
        filled += take
    return out


def _antennas_y27() -> np.ndarray:
    """27 antennas on a generic three-arm power-law 'Y' (9 per arm, 120 deg apart,
    radius ~ i^1.716): (east, north) in arbitrary units.  Not a real array."""
    pos = []
    for arm in range(3):
        az = math.radians(5.0 + 120.0 * arm)
        for i in range(1, 10):
            r = float(i) ** 1.716
            pos.append((r * math.sin(az), r * math.cos(az)))
    return np.asarray(pos)


def _antennas_ska197(seed: int) -> np.ndarray:
    """197 antennas, 'SKA-like random': 98 in a Gaussian core (sigma 1) + 99 with
    log-uniform radius in [1, 60] and uniform azimuth.  (east, north)."""
    rng = rng_for(seed, STREAM_UV)
    core = rng.standard_normal((98, 2))
    r = np.exp(rng.uniform(0.0, math.log(60.0), size=99))
    az = rng.uniform(0.0, 2 * math.pi, size=99)
    outer = np.stack([r * np.sin(az), r * np.cos(az)], axis=1)
    return np.concatenate([core, outer], axis=0)


def uv_rotation_synthesis(ant_en: np.ndarray, lat_deg: float, dec_deg: float, n_chan: int,
                          M: int, K: int, dtype: str, hours: float = 8.0, step_s: float = 10.0,
                          fill: float = 0.8) -> np.ndarray:
    """Rotation-synthesis tracks ([35]-style geometry): baselines
    (E, N) -> (Lx, Ly, Lz) = (-N sin(lat), E, N cos(lat)); for hour angle H:
    u = Lx sin H + Ly cos H; v = -Lx sin(dec) cos H + Ly sin(dec) sin H + Lz cos(dec).
    Order is time-major: (time, channel, baseline).  Channel c scales uv by 1 + 0.01 c.
    One global scale so that max(|u|,|v|) = fill * K/2.  First M samples kept."""
    lat, dec = math.radians(lat_deg), math.radians(dec_deg)
    i, j = np.triu_indices(len(ant_en), k=1)
    E = ant_en[i, 0] - ant_en[j, 0]
    N = ant_en[i, 1] - ant_en[j, 1]
    Lx, Ly, Lz = -N * math.sin(lat), E, N * math.cos(lat)
    n_t = int(round(hours * 3600.0 / step_s))
    H = np.radians((-hours / 2 + hours * (np.arange(n_t) + 0.5) / n_t) * 15.0)
    chan = 1.0 + 0.01 * np.arange(n_chan)
    nb = len(E)
    # global scale from the extreme (largest channel) without materialising everything
    umax = 0.0
    for h in (H[:: max(1, n_t // 64)].tolist() + [H[-1]]):
        u = Lx * math.sin(h) + Ly * math.cos(h)
        v = -Lx * math.sin(dec) * math.cos(h) + Ly * math.sin(dec) * math.sin(h) + Lz * math.cos(dec)
        umax = max(umax, float(np.abs(u).max()), float(np.abs(v).max()))
    # exact max over all steps (cheap: n_t x nb reductions, done in blocks)
    for t0 in range(0, n_t, 256):
        h = H[t0:t0 + 256, None]
        u = Lx[None, :] * np.sin(h) + Ly[None, :] * np.cos(h)
        v = (-Lx[None, :] * math.sin(dec) * np.cos(h) + Ly[None, :] * math.sin(dec) * np.sin(h)
             + Lz[None, :] * math.cos(dec))
        umax = max(umax, float(np.abs(u).max()), float(np.abs(v).max()))
    scale = fill * (K / 2) / (umax * chan[-1])
    rd = real_dtype(dtype)
    out = np.empty((M, 2), dtype=rd)
    filled = 0
    for t in range(n_t):
        if filled >= M:
            break
        h = H[t]
        u = (Lx * math.sin(h) + Ly * math.cos(h)) * scale
        v = (-Lx * math.sin(dec) * math.cos(h) + Ly * math.sin(dec) * math.sin(h)
             + Lz * math.cos(dec)) * scale
        blk = np.empty((n_chan, nb, 2), dtype=np.float64)
        blk[:, :, 0] = chan[:, None] * u[None, :]
        blk[:, :, 1] = chan[:, None] * v[None, :]
        blk = blk.reshape(-1, 2)
        take = min(len(blk), M - filled)
        out[filled:filled + take] = blk[:take].astype(rd)
        filled += take
    if filled < M:
        raise ValueError(f"rotation synthesis produced only {filled} < M={M} samples")
    return out


def make_uv(cfg: Config, M: int | None = None, J: int | None = None) -> np.ndarray:
    """(u, v) for a config; M / J may be overridden (bounded samples, J=8 variant)."""
    M = cfg.M if M is None else int(M)
    J = cfg.J if J is None else int(J)
    if cfg.uv == "gauss":
        return uv_gaussian(M, cfg.K, J, cfg.sigma_div, cfg.seed, cfg.dtype)
    if cfg.uv == "vla27":
        return uv_rotation_synthesis(_antennas_y27(), 34.0, 60.0, 10, M, cfg.K, cfg.dtype)
    if cfg.uv == "ska197":
        return uv_rotation_synthesis(_antennas_ska197(cfg.seed), -30.0, -60.0, 9, M, cfg.K, cfg.dtype)
    raise ValueError(cfg.uv)


def shuffle_order(M: int, seed: int) -> np.ndarray:
    """Seeded permutation (BASELINE.json configs[2]: 'time-ordered and shuffled')."""
    return rng_for(seed, STREAM_SHUFFLE).permutation(M)


# --------------------------------------------------------------------------- weights / noise
def make_weights(cfg: Config, M: int | None = None) -> np.ndarray:
    M = cfg.M if M is None else int(M)
    rd = real_dtype(cfg.dtype)
    if cfg.weights == "unit":
        return np.ones(M, dtype=rd)
    return rng_for(cfg.seed, STREAM_W).uniform(0.5, 1.5, size=M).astype(rd)


def add_noise(y: np.ndarray, snr_db: float, seed: int) -> np.ndarray:
    """y + n, n_k = sigma (xi1 + i xi2)/sqrt(2), sigma = ||y||/sqrt(M) 10^(-snr/20)
    (BASELINE.json configs[1] '30 dB input SNR')."""
    rng = rng_for(seed, STREAM_NOISE)
    M = y.shape[0]
    sigma = float(np.linalg.norm(y)) / math.sqrt(M) * 10.0 ** (-snr_db / 20.0)
    nz = (rng.standard_normal(M) + 1j * rng.standard_normal(M)) * (sigma / math.sqrt(2.0))
    return (y + nz).astype(y.dtype)


def make_problem(index: int, M: int | None = None, J: int | None = None):
    """(cfg, x, uv, w) for config `index`, optionally with a bounded M."""
    cfg = CONFIGS[index]
    x = make_image(cfg.n, cfg.seed, cfg.dtype)
    uv = make_uv(cfg, M, J)
    w = make_weights(cfg, M)
    return cfg, x, uv, w
