"""The five BASELINE.json workloads as concrete, seeded recipes.

Nothing here is reconstruction arithmetic: only optics constants, LED layouts and
the recipe of the ground-truth pupil / object / noise for each config.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Sequence, Tuple

import numpy as np

CONFIG_NAMES = ("cfg0_smoke64", "cfg1_single256", "cfg2_batch64_256",
                "cfg3_batch1024_512", "cfg4_slide20000_256")


@dataclasses.dataclass(frozen=True)
class ApicConfig:
    index: int
    name: str
    tile_n: int                     # N, raw tile side (512 px patches)
    upsample: int                   # u, output grid = u*N
    wavelength_um: float            # PAPER.md:153 (green LED ~0.52 um)
    pixel_um: float                 # 3.45 um pitch / 10x
    na_obj: float                   # 10x / 0.25 NA
    n_bright: int                   # NA-matching LEDs on the NA_obj ring
    dark_rings: Tuple[Tuple[float, int], ...]   # (NA_ill, count) per darkfield ring, ascending NA
    noll_truth: Tuple[int, ...]     # Noll indices present in the ground-truth pupil
    noll_fit: Tuple[int, ...]       # Noll indices the reconstruction fits (>= 4)
    pupil_recipe: str               # "uniform" | "norm" | "field"
    pupil_strength: float           # U(-s, s) rad | ||c||_2 = s rad | max-over-tiles ||c||_2 = s rad
    amp_range: Tuple[float, float]
    phase_range: Tuple[float, float]
    noise: str                      # "none" | "gauss" | "poisson"
    batch: int
    grid: Tuple[int, int]           # tile grid (gx, gy) for field-dependent pupils
    background_fraction: float      # share of blank tiles (cfg 4)
    seed_base: int

    @property
    def n_dark(self) -> int:
        return sum(n for _, n in self.dark_rings)

    @property
    def out_n(self) -> int:
        return self.tile_n * self.upsample

    @property
    def pupil_radius_bins(self) -> float:
        """R = NA * N * dx / lambda (SURVEY §8 notation)."""
        return self.na_obj * self.tile_n * self.pixel_um / self.wavelength_um


def _mk(index, **kw) -> ApicConfig:
    base = dict(wavelength_um=0.52, pixel_um=0.345, na_obj=0.25, grid=(1, 1),
                background_fraction=0.0, seed_base=1000 * index)
    base.update(kw)
    return ApicConfig(index=index, name=CONFIG_NAMES[index], **base)


_RINGS_24 = ((0.30, 8), (0.40, 8))
_RINGS_44 = ((0.28, 8), (0.34, 12), (0.45, 12))

_CONFIGS = {
    0: _mk(0, tile_n=64, upsample=2, n_bright=4, dark_rings=(),
           noll_truth=(4, 5, 6), noll_fit=(4, 5, 6), pupil_recipe="uniform", pupil_strength=1.0,
           amp_range=(0.8, 1.0), phase_range=(0.0, math.pi / 2), noise="none", batch=1),
    1: _mk(1, tile_n=256, upsample=2, n_bright=8, dark_rings=(),
           noll_truth=tuple(range(2, 17)), noll_fit=tuple(range(4, 17)), pupil_recipe="norm",
           pupil_strength=0.5, amp_range=(0.8, 1.0), phase_range=(0.0, math.pi / 2),
           noise="gauss", batch=1),
    2: _mk(2, tile_n=256, upsample=3, n_bright=8, dark_rings=_RINGS_24,
           noll_truth=tuple(range(2, 17)), noll_fit=tuple(range(4, 17)), pupil_recipe="field",
           pupil_strength=0.5, amp_range=(0.8, 1.0), phase_range=(0.0, math.pi / 2),
           noise="poisson", batch=64, grid=(8, 8)),
    3: _mk(3, tile_n=512, upsample=3, n_bright=12, dark_rings=_RINGS_44,
           noll_truth=tuple(range(2, 38)), noll_fit=tuple(range(4, 38)), pupil_recipe="norm",
           pupil_strength=1.0, amp_range=(0.6, 1.0), phase_range=(0.0, math.pi),
           noise="poisson", batch=1024),
    4: _mk(4, tile_n=256, upsample=3, n_bright=8, dark_rings=_RINGS_24,
           noll_truth=tuple(range(2, 17)), noll_fit=tuple(range(4, 17)), pupil_recipe="field",
           pupil_strength=0.5, amp_range=(0.8, 1.0), phase_range=(0.0, math.pi / 2),
           noise="poisson", batch=20000, grid=(200, 100), background_fraction=0.4),
}


def get_config(index: int, **overrides) -> ApicConfig:
    """Config ``index`` of BASELINE.json; ``overrides`` make reduced variants for quick tests
    (e.g. ``get_config(2, tile_n=64, batch=4, grid=(2, 2))``)."""
    cfg = _CONFIGS[index]
    return dataclasses.replace(cfg, **overrides) if overrides else cfg


def led_kvectors(cfg: ApicConfig) -> Tuple[np.ndarray, np.ndarray]:
    """Transverse illumination k-vectors in cycles/um, SURVEY R20 layout.

    NA-matching LEDs: azimuth 360*i/n on the NA_obj ring.  Darkfield ring r (ascending NA):
    azimuth 360*(i + 0.5*(r mod 2))/n_r.  Returns (k_bright [n_b,2], k_dark [n_d,2]) as (kx, ky).
    """
    lam = cfg.wavelength_um
    kb = np.zeros((cfg.n_bright, 2))
    for i in range(cfg.n_bright):
        a = 2.0 * math.pi * i / cfg.n_bright
        kb[i] = (cfg.na_obj / lam * math.cos(a), cfg.na_obj / lam * math.sin(a))
    kd: List[Sequence[float]] = []
    for r, (na, n) in enumerate(cfg.dark_rings):
        for i in range(n):
            a = 2.0 * math.pi * (i + 0.5 * (r % 2)) / n
            kd.append((na / lam * math.cos(a), na / lam * math.sin(a)))
    return kb, np.asarray(kd, dtype=np.float64).reshape(-1, 2)


def plan_args(cfg: ApicConfig) -> tuple:
    """Positional arguments of the library's plan constructor for this recipe: (N, u, lambda, pixel, NA,
    k_bright, k_dark, fitted Noll indices) - the optics and LED layout only, no method arithmetic."""
    kb, kd = led_kvectors(cfg)
    return (cfg.tile_n, cfg.upsample, cfg.wavelength_um, cfg.pixel_um, cfg.na_obj, kb, kd, tuple(cfg.noll_fit))
