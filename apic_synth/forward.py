"""Forward model and noise: synthetic intensity stacks shaped like the paper's tiles.

Model (Eq. 1-2, written in the DC-centred frame of Eq. 3, PAPER.md:76-80;
SURVEY.md R2): with integer frequency bins k on the raw N x N grid, kappa_i = k_i*N*dx (bins)
and R = NA*N*dx/lambda,

    S'_i(k) = O(k) * 1[|k + kappa_i| <= R] * exp(j*phi(k + kappa_i)),
    I_i(m)  = | sum_k S'_i(k) exp(+j 2 pi k.m / N) |^2 ,   m in [0, N)^2 .

O(k) are the Fourier coefficients of the object sampled on the (uN)^2 output grid
(o(X) = sum_k O(k) exp(+j 2 pi k.X/(uN))), so raw pixel m sits at output pixel u*m.

The ground-truth pupil phase phi = sum_j c_j Z_j uses Noll-ordered Zernike polynomials that
are evaluated HERE through Jacobi polynomials (scipy) - deliberately a different formula from
the oracle's and the CUDA plan's, so that coefficient recovery is a real cross-check.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Iterable, List, Optional, Tuple

import numpy as np
from scipy.special import eval_jacobi

from .configs import ApicConfig, led_kvectors

_DISC_RTOL = 1e-9          # inclusive disc test |k+kappa|^2 <= R^2 (1+1e-9)


# ----------------------------------------------------------------------------------------------
# Ground-truth Zernike (Noll order) via enumeration + Jacobi polynomials
# ----------------------------------------------------------------------------------------------
def noll_table(jmax: int) -> Dict[int, Tuple[int, int]]:
    """Noll j -> (n, m) by enumeration: radial order n ascending, |m| ascending within n,
    even j <-> cosine (m > 0), odd j <-> sine (m < 0)."""
    table: Dict[int, Tuple[int, int]] = {}
    j = 1
    n = 0
    while j <= jmax:
        for am in range(n % 2, n + 1, 2):
            if am == 0:
                table[j] = (n, 0)
                j += 1
            else:
                for jj in (j, j + 1):
                    table[jj] = (n, am if jj % 2 == 0 else -am)
                j += 2
        n += 1
    return table


def truth_zernike(j: int, x: np.ndarray, y: np.ndarray) -> np.ndarray:
    """Z_j at Cartesian pupil coordinates (x, y) = (k + kappa)/R; unit RMS on the unit disc."""
    n, m = noll_table(j)[j]
    am = abs(m)
    rho = np.hypot(x, y)
    th = np.arctan2(y, x)
    s = (n - am) // 2
    radial = (-1.0) ** s * rho ** am * eval_jacobi(s, am, 0, 1.0 - 2.0 * rho * rho)
    if m == 0:
        return math.sqrt(n + 1.0) * radial
    ang = np.cos(am * th) if m > 0 else np.sin(am * th)
    return math.sqrt(2.0 * (n + 1.0)) * radial * ang


# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass
class TileTruth:
    tile: int
    blank: bool
    coef: Dict[int, float]            # Noll index -> rad (ground-truth pupil)
    obj: np.ndarray                   # complex128 [uN][uN] object on the output grid
    gain_bright: float = 1.0          # photons per intensity unit (poisson); 1 otherwise
    gain_dark: float = 1.0
    clean: Optional[np.ndarray] = None    # noise-free fp64 stack (only if keep_clean)


def bins_fft_order(n: int) -> np.ndarray:
    """Signed integer frequency bins in numpy FFT order: 0..n/2-1, -n/2..-1."""
    return np.rint(np.fft.fftfreq(n) * n).astype(np.int64)


def make_object(cfg: ApicConfig, rng: np.random.Generator, blank: bool = False) -> np.ndarray:
    """amplitude i.i.d. U[lo,hi] per output pixel; phase = white Gaussian noise,
    periodic Gaussian filter sigma = 3 output px, min-max rescaled to the stated range."""
    nh = cfg.out_n
    if blank:
        return np.ones((nh, nh), dtype=np.complex128)
    amp = rng.uniform(cfg.amp_range[0], cfg.amp_range[1], size=(nh, nh))
    w = rng.standard_normal((nh, nh))
    f = np.fft.fftfreq(nh)
    sigma = 3.0
    g = np.exp(-2.0 * (math.pi * sigma) ** 2 * (f[None, :] ** 2 + f[:, None] ** 2))
    p = np.real(np.fft.ifft2(np.fft.fft2(w) * g))
    p = (p - p.min()) / (p.max() - p.min())
    ph = cfg.phase_range[0] + (cfg.phase_range[1] - cfg.phase_range[0]) * p
    return amp * np.exp(1j * ph)


def _tile_xy(cfg: ApicConfig, tile: int) -> Tuple[float, float]:
    gx, gy = cfg.grid
    tx, ty = tile % gx, (tile // gx) % gy
    return (-1.0 + (2.0 * tx + 1.0) / gx, -1.0 + (2.0 * ty + 1.0) / gy)


def _field_poly(cfg: ApicConfig) -> np.ndarray:
    """q[j, 6]: seeded quadratic field dependence, scaled so that max over the tile grid of
    ||c||_2 equals cfg.pupil_strength."""
    rng = np.random.default_rng(cfg.seed_base + 10 ** 6)
    q = rng.standard_normal((len(cfg.noll_truth), 6))
    gx, gy = cfg.grid
    xs = -1.0 + (2.0 * np.arange(gx) + 1.0) / gx
    ys = -1.0 + (2.0 * np.arange(gy) + 1.0) / gy
    X, Y = np.meshgrid(xs, ys, indexing="xy")
    basis = np.stack([np.ones_like(X), X, Y, X * X, X * Y, Y * Y], axis=0)   # a+b<=2
    c = np.tensordot(q, basis, axes=(1, 0))                                   # [j, gy, gx]
    worst = np.sqrt((c ** 2).sum(axis=0)).max()
    return q * (cfg.pupil_strength / worst)


def truth_coefficients(cfg: ApicConfig, tile: int, rng: np.random.Generator) -> Dict[int, float]:
    nt = len(cfg.noll_truth)
    if cfg.pupil_recipe == "uniform":
        c = rng.uniform(-cfg.pupil_strength, cfg.pupil_strength, size=nt)
    elif cfg.pupil_recipe == "norm":
        c = rng.standard_normal(nt)
        c *= cfg.pupil_strength / np.linalg.norm(c)
    elif cfg.pupil_recipe == "field":
        q = _field_poly(cfg)
        x, y = _tile_xy(cfg, tile)
        c = q @ np.array([1.0, x, y, x * x, x * y, y * y])
        rng.standard_normal(nt)            # keep the per-tile stream aligned across recipes
    else:
        raise ValueError(cfg.pupil_recipe)
    return {j: float(v) for j, v in zip(cfg.noll_truth, c)}


def blank_flags(cfg: ApicConfig) -> np.ndarray:
    """Which tiles of the config are background (amp 1, phase 0); seeded, cfg 4 only."""
    if cfg.background_fraction <= 0.0:
        return np.zeros(cfg.batch, dtype=bool)
    rng = np.random.default_rng(cfg.seed_base + 2 * 10 ** 6)
    return rng.random(cfg.batch) < cfg.background_fraction


def object_spectrum_raw(cfg: ApicConfig, obj: np.ndarray) -> np.ndarray:
    """O(k) on the raw grid's integer bins, FFT order [N][N] (ky, kx); DC = spatial mean."""
    nh, n = cfg.out_n, cfg.tile_n
    oh = np.fft.fft2(obj) / float(nh * nh)
    k = bins_fft_order(n)
    idx = np.mod(k, nh)
    return oh[np.ix_(idx, idx)]


def pupil_phase_at(cfg: ApicConfig, coef: Dict[int, float], kap: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """(disc mask, phi(k + kappa)) on the raw grid's bins, FFT order."""
    n = cfg.tile_n
    r = cfg.pupil_radius_bins
    k = bins_fft_order(n).astype(np.float64)
    px = (k[None, :] + kap[0]) / r
    py = (k[:, None] + kap[1]) / r
    px, py = np.broadcast_arrays(px, py)
    mask = (px * px + py * py) <= (1.0 + _DISC_RTOL)
    phi = np.zeros((n, n))
    for j, c in coef.items():
        if c != 0.0:
            phi += c * truth_zernike(j, px, py)
    return mask, phi


def forward_stack(cfg: ApicConfig, obj: np.ndarray, coef: Dict[int, float]) -> np.ndarray:
    """Noise-free fp64 intensities [n_bright + n_dark][N][N]; NA-matching images first."""
    n = cfg.tile_n
    kb, kd = led_kvectors(cfg)
    scale = n * cfg.pixel_um                       # kappa = k * N * dx
    o_raw = object_spectrum_raw(cfg, obj)
    out = np.empty((cfg.n_bright + cfg.n_dark, n, n))
    for i, kvec in enumerate(list(kb) + list(kd)):
        kap = np.asarray(kvec) * scale
        mask, phi = pupil_phase_at(cfg, coef, kap)
        s = np.where(mask, o_raw * np.exp(1j * phi), 0.0)
        field = np.fft.ifft2(s) * float(n * n)
        out[i] = field.real ** 2 + field.imag ** 2
    return out


def add_noise(cfg: ApicConfig, clean: np.ndarray, rng: np.random.Generator,
              truth: TileTruth) -> np.ndarray:
    """SURVEY R21.  Returns the fp32 stack the reconstruction sees."""
    nb = cfg.n_bright
    if cfg.noise == "none":
        return clean.astype(np.float32)
    if cfg.noise == "gauss":
        sigma = 0.005 * clean.mean()
        return (clean + sigma * rng.standard_normal(clean.shape)).astype(np.float32)
    if cfg.noise == "poisson":
        out = np.empty(clean.shape, dtype=np.float32)
        g_b = 5000.0 / clean[:nb].mean()
        raw = np.minimum(rng.poisson(g_b * clean[:nb]), 65535).astype(np.uint16)
        out[:nb] = raw.astype(np.float64) / g_b
        truth.gain_bright = g_b
        if clean.shape[0] > nb:
            m_d = clean[nb:].mean()
            g_d = 500.0 / m_d if m_d > 0 else 1.0
            rawd = np.minimum(rng.poisson(g_d * clean[nb:]), 65535).astype(np.uint16)
            out[nb:] = rawd.astype(np.float64) / g_d
            truth.gain_dark = g_d
        return out
    raise ValueError(cfg.noise)


def make_tile(cfg: ApicConfig, tile: int = 0, *, noise: Optional[str] = None,
              blank: Optional[bool] = None, keep_clean: bool = False
              ) -> Tuple[np.ndarray, TileTruth]:
    """One tile's fp32 intensity stack [n_bright+n_dark][N][N] and its ground truth.

    Seed = cfg.seed_base + tile; draw order: amplitude, phase noise, pupil
    coefficients, measurement noise.
    """
    if noise is not None:
        cfg = dataclasses.replace(cfg, noise=noise)
    rng = np.random.default_rng(cfg.seed_base + tile)
    if blank is None:
        blank = bool(blank_flags(cfg)[tile]) if cfg.background_fraction > 0 else False
    obj = make_object(cfg, rng, blank=blank)
    coef = truth_coefficients(cfg, tile, rng)
    truth = TileTruth(tile=tile, blank=blank, coef=coef, obj=obj)
    clean = forward_stack(cfg, obj, coef)
    if keep_clean:
        truth.clean = clean
    stack = add_noise(cfg, clean, rng, truth)
    return stack, truth


def make_batch(cfg: ApicConfig, tiles: Iterable[int], **kw) -> Tuple[np.ndarray, List[TileTruth]]:
    tiles = list(tiles)
    n = cfg.tile_n
    out = np.empty((len(tiles), cfg.n_bright + cfg.n_dark, n, n), dtype=np.float32)
    truths: List[TileTruth] = []
    for b, t in enumerate(tiles):
        out[b], tr = make_tile(cfg, t, **kw)
        truths.append(tr)
    return out, truths
