"""On-device generator of the slide-scale workload (BASELINE.json config 4: "20,000 tiles ... generated on
device from a seed").

Same recipe as ``forward.py`` (object on the (uN)^2 grid, object-frame forward model of PAPER.md Eq. 1-3,
Poisson noise at 5000 / 500 mean photons, uint16 counts) written with torch tensor operations so that a batch of
tiles is produced directly in HBM; the random numbers come from torch's counter-based (Philox) CUDA generator,
seeded per tile with (seed, tile index), so a tile's stack does not depend on how the slide is cut into
batches - up to last-bit effects of the batched library FFT (a count differs by one in < 0.01 % of the pixels).  This is INPUT SYNTHESIS for tests and bench.py only: no reconstruction arithmetic, no import of
``oracle`` or of the CUDA library; the ground-truth Zernike tables are evaluated once on the host by
``forward.truth_zernike`` (Jacobi polynomials) and uploaded.

The numbers differ from ``forward.make_tile`` (another RNG, fp32 transforms), which is fine: parity tests read the
generated stacks back and give the very same values to the oracle.
"""
from __future__ import annotations

import math
from typing import Tuple

import numpy as np

from .configs import ApicConfig, led_kvectors
from .forward import _DISC_RTOL, _field_poly, bins_fft_order, blank_flags, truth_zernike


class DeviceGenerator:
    def __init__(self, cfg: ApicConfig, device="cuda", seed: int | None = None):
        import torch
        self.torch = torch
        self.cfg = cfg
        self.device = torch.device(device)
        self.seed = int(cfg.seed_base if seed is None else seed)
        n, r = cfg.tile_n, cfg.pupil_radius_bins
        kb, kd = led_kvectors(cfg)
        k = bins_fft_order(n).astype(np.float64)
        masks, basis = [], []
        for kvec in list(kb) + list(kd):
            kap = np.asarray(kvec) * (n * cfg.pixel_um)
            px, py = np.broadcast_arrays((k[None, :] + kap[0]) / r, (k[:, None] + kap[1]) / r)
            masks.append((px * px + py * py) <= (1.0 + _DISC_RTOL))
            basis.append(np.stack([truth_zernike(j, px, py) for j in cfg.noll_truth]))
        self.mask = torch.from_numpy(np.stack(masks)).to(self.device)                      # [L][N][N] bool
        self.basis = torch.from_numpy(np.stack(basis).astype(np.float32)).to(self.device)   # [L][J][N][N]
        self.q = torch.from_numpy(_field_poly(cfg).astype(np.float32)).to(self.device)      # [J][6]
        self.blank = blank_flags(cfg)                                                       # host bool [batch]
        nh = cfg.out_n
        f = np.fft.fftfreq(nh)
        g = np.exp(-2.0 * (math.pi * 3.0) ** 2 * (f[None, :] ** 2 + f[:, None] ** 2))
        self.gauss = torch.from_numpy(g.astype(np.float32)).to(self.device)
        idx = np.mod(bins_fft_order(n), nh)
        self.crop = torch.from_numpy(idx).to(self.device)

    def tile_xy(self, tiles: np.ndarray) -> np.ndarray:
        gx, gy = self.cfg.grid
        tx, ty = tiles % gx, (tiles // gx) % gy
        return np.stack([-1.0 + (2.0 * tx + 1.0) / gx, -1.0 + (2.0 * ty + 1.0) / gy], axis=1)

    def coefficients(self, tiles: np.ndarray):
        """Ground-truth Zernike coefficients [B][J] (slide-wide quadratic field dependence)."""
        torch = self.torch
        xy = self.tile_xy(np.asarray(tiles))
        x, y = xy[:, 0], xy[:, 1]
        mono = np.stack([np.ones_like(x), x, y, x * x, x * y, y * y], axis=1).astype(np.float32)
        return torch.from_numpy(mono).to(self.device) @ self.q.T

    def generate(self, tile0: int, count: int) -> Tuple["torch.Tensor", "torch.Tensor", np.ndarray]:
        """Tiles tile0 .. tile0+count-1 -> (raw uint16 [B][n_img][N][N], scale float32 [B][n_img], blank bool [B]).
        intensity = count * scale, in the common radiometric units of DESIGN.md R17."""
        torch = self.torch
        cfg, dev = self.cfg, self.device
        nh, n, nb = cfg.out_n, cfg.tile_n, cfg.n_bright
        tiles = np.arange(tile0, tile0 + count)
        blank = self.blank[tiles]
        gen = torch.Generator(device=dev)
        amp = torch.empty((count, nh, nh), device=dev)
        w = torch.empty((count, nh, nh), device=dev)
        for b, t in enumerate(tiles):
            gen.manual_seed((self.seed << 24) + int(t))
            amp[b].uniform_(cfg.amp_range[0], cfg.amp_range[1], generator=gen)
            w[b].normal_(generator=gen)
        p = torch.fft.ifft2(torch.fft.fft2(w) * self.gauss).real
        lo = p.amin(dim=(1, 2), keepdim=True)
        hi = p.amax(dim=(1, 2), keepdim=True)
        ph = cfg.phase_range[0] + (cfg.phase_range[1] - cfg.phase_range[0]) * (p - lo) / (hi - lo)
        obj = torch.polar(amp, ph)
        bl = torch.from_numpy(blank).to(dev)
        obj[bl] = 1.0
        oh = torch.fft.fft2(obj) / float(nh * nh)
        o_raw = oh[:, self.crop][:, :, self.crop]                                           # [B][N][N], FFT order
        coef = self.coefficients(tiles)                                                     # [B][J]
        phi = torch.einsum("bj,ljyx->blyx", coef, self.basis)                               # [B][L][N][N]
        s = torch.where(self.mask[None], o_raw[:, None] * torch.polar(torch.ones_like(phi), phi), torch.zeros((), device=dev, dtype=o_raw.dtype))
        field = torch.fft.ifft2(s) * float(n * n)
        clean = field.real ** 2 + field.imag ** 2                                           # [B][L][N][N]
        del s, field, phi
        m_b = clean[:, :nb].mean(dim=(1, 2, 3))
        m_d = clean[:, nb:].mean(dim=(1, 2, 3)) if clean.shape[1] > nb else torch.ones_like(m_b)
        g_b = 5000.0 / m_b
        g_d = torch.where(m_d > 1e-9, 500.0 / m_d.clamp_min(1e-30), torch.ones_like(m_d))
        gain = torch.cat([g_b[:, None].expand(-1, nb), g_d[:, None].expand(-1, clean.shape[1] - nb)], dim=1)   # [B][L]
        raw = torch.empty(clean.shape, device=dev, dtype=torch.uint16)
        for b, t in enumerate(tiles):
            gen.manual_seed((self.seed << 24) + (1 << 23) + int(t))
            cnt = torch.poisson(clean[b] * gain[b][:, None, None], generator=gen)
            raw[b] = cnt.clamp_(max=65535.0).to(torch.uint16)
        scale = (1.0 / gain).to(torch.float32).contiguous()
        return raw, scale, blank
