"""fp64 CPU oracle of the within-FOV reassembly of overlapping tiles.

TEST INFRASTRUCTURE - not part of the product path; shares no code with the CUDA library.

What the paper fixes: a field of view is cut into patches that are "individually reconstructed and then stitched
together"; between fields of view "the overlapping regions were blended to smoothen any visible
seams" and the assembly proceeds from the top-left corner against the regions already stitched.
BASELINE.json config 4 gives the tiles "10 % spatial overlap".  The paper states neither the blend nor what happens to
a complex field's global phase, so the readings are (B6-B8):

  B6  geometry: tiles_y x tiles_x tiles of T x T output pixels on a regular grid with `overlap` pixels shared between
      neighbours, 0 <= 2 overlap <= T; tile (r, c) covers FOV rows r (T - overlap) ... r (T - overlap) + T - 1.
  B7  blend: linear and separable.  Inside an overlap of width v the weight of the tile further right (down) is
      (k + 1/2) / v at the overlap's k-th pixel and that of the other tile is 1 minus it; outside overlaps a tile's
      weight is 1.  The weights of the tiles that cover a pixel sum to 1 exactly.
  B8  global phase: every tile comes out of the reconstruction with its own DC real-positive (R14), i.e. multiplied
      by an unknown unit factor relative to its neighbours.  Tiles are brought to the phase of tile (0, 0) in raster
      order against their already aligned left and upper neighbours (the order of PAPER.md:149):
          u(0,0) = 1,   u(t) = c / |c|,   c = u(left) C_h(t) + u(up) C_v(t),
          C_h(t) = sum over the overlap with the left neighbour of  f_left conj f_t   (C_v likewise, upper neighbour),
      and the FOV is  sum_t w_t u_t f_t.  align = False skips B8 (u = 1).  |c| = 0 (blank overlaps) gives u = 1.

Pins (tests/test_oracle_reassemble.py, -m "not gpu"): weights sum to 1 and reproduce a hand-computed 1-D ramp; tiles
cut from a known FOV and multiplied by arbitrary unit factors reassemble to that FOV times conj(factor of tile (0,0))
to 1e-12; overlap 0 is plain tiling; identical constant tiles give the constant; a brute-force per-pixel double loop
on a tiny case equals the vectorised form.
"""
from __future__ import annotations

import numpy as np


def fov_size(tiles: int, t: int, overlap: int) -> int:
    """B6: extent of `tiles` tiles of `t` pixels sharing `overlap` pixels with each neighbour."""
    return tiles * (t - overlap) + overlap


def ramp_weights(t: int, overlap: int, first: bool, last: bool) -> np.ndarray:
    """B7: 1-D weight of a tile along one axis; `first` / `last`: the tile has no neighbour before / after it."""
    w = np.ones(t, dtype=np.float64)
    if overlap > 0:
        r = (np.arange(overlap, dtype=np.float64) + 0.5) / overlap
        if not first:
            w[:overlap] = r                 # this tile is the one "further right": its weight rises
        if not last:
            w[t - overlap:] = 1.0 - r       # and falls where the next tile takes over
    return w


def pair_correlations(fields: np.ndarray, overlap: int):
    """B8: C_h[r, c] = sum over the overlap with the left neighbour of f_left conj f, C_v likewise (0 without one)."""
    ty, tx, t, _ = fields.shape
    ch = np.zeros((ty, tx), dtype=np.complex128)
    cv = np.zeros((ty, tx), dtype=np.complex128)
    if overlap == 0:
        return ch, cv
    f = fields.astype(np.complex128)
    for r in range(ty):
        for c in range(tx):
            if c > 0:
                ch[r, c] = np.sum(f[r, c - 1][:, t - overlap:] * np.conj(f[r, c][:, :overlap]))
            if r > 0:
                cv[r, c] = np.sum(f[r - 1, c][t - overlap:, :] * np.conj(f[r, c][:overlap, :]))
    return ch, cv


def phase_factors(ch: np.ndarray, cv: np.ndarray) -> np.ndarray:
    """B8: unit factors u in raster order."""
    ty, tx = ch.shape
    u = np.ones((ty, tx), dtype=np.complex128)
    for r in range(ty):
        for c in range(tx):
            if r == 0 and c == 0:
                continue
            acc = 0.0 + 0.0j
            if c > 0:
                acc += u[r, c - 1] * ch[r, c]
            if r > 0:
                acc += u[r - 1, c] * cv[r, c]
            u[r, c] = acc / abs(acc) if abs(acc) > 0.0 else 1.0
    return u


def reassemble(fields: np.ndarray, overlap: int, align: bool = True):
    """fields: [tiles_y][tiles_x][T][T] complex.  Returns (fov [H][W] complex128, u [tiles_y][tiles_x])."""
    ty, tx, t, t2 = fields.shape
    if t != t2 or overlap < 0 or 2 * overlap > t:
        raise ValueError("bad tile geometry")
    f = fields.astype(np.complex128)
    u = phase_factors(*pair_correlations(f, overlap)) if align else np.ones((ty, tx), dtype=np.complex128)
    step = t - overlap
    out = np.zeros((fov_size(ty, t, overlap), fov_size(tx, t, overlap)), dtype=np.complex128)
    for r in range(ty):
        wy = ramp_weights(t, overlap, r == 0, r == ty - 1)
        for c in range(tx):
            wx = ramp_weights(t, overlap, c == 0, c == tx - 1)
            out[r * step:r * step + t, c * step:c * step + t] += (wy[:, None] * wx[None, :]) * (u[r, c] * f[r, c])
    return out, u
