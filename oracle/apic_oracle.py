"""Plain, slow, fp64 CPU oracle of the APIC closed-form reconstruction (numpy).

TEST INFRASTRUCTURE - not part of the product path; shares no code with the CUDA library.
Every function cites the passage of /root/reference/PAPER.md it follows ("PAPER.md:<line>")
and, where the paper is silent or garbled, the reading taken (R-numbers of SURVEY.md §8(c),
restated in DESIGN.md §3).

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``):
  fft2n / ifft2u ........ naive O(N^4) DFT at N=64, Parseval, round trip
  zernike ............... Noll (n,m) table of the literature for j<=15, closed forms Z4/Z5/Z11,
                          orthonormality on the unit disc by quadrature
  kk_field .............. exact recovery of S'_i e^{-j arg DC} from noise-free forward data,
                          error decay with kk_pad 1 -> 2 -> 4 (aliasing of log harmonics only)
  aberration_* .......... closed form for pure defocus (beta linear in K), zero piston/tilt
                          columns, row counts of SURVEY §8(c), exact c from true spectra
  stitch ................ equals the true object spectrum on the union of discs
  darkfield_* ........... with the exact known spectrum the solved unknown spectrum equals the
                          truth; FFT correlation == direct double sum; index-set sizes
  reconstruct ........... noise-free end-to-end agreement with the ground-truth object
PARITY UNPINNED: behaviour on real, non-periodic tiles (edge leakage, NA mismatch, LED
mis-calibration) - no such data exists in the container.

Conventions (O0 / R1): arrays are [y][x]; spatial origin at index 0; forward transform
S[k] = sum_x s[x] exp(-j 2 pi k.x / N); spectra are stored divided by N^2 (DC = mean), on
signed integer bins k in [-N/2, N/2), in numpy FFT order unless a name says "centred".
R = NA*N*dx/lambda (bins), kappa_i = k_i*N*dx (bins, real valued).
"""
from __future__ import annotations

import dataclasses
import itertools
import math
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

TWO_PI = 2.0 * math.pi
DISC_RTOL = 1e-9            # R3: inclusive disc test |k+kappa|^2 <= R^2 (1 + 1e-9)
HALFPLANE_TAU = 1e-4        # R5: |k.kappa/|kappa|| <= tau bins counts as "on the line"
KAPPA_ORDER_QUANTUM = 1e-6  # R15: |kappa| compared after rounding to 1e-6 bins (ties: input order)
MAX_UNKNOWN_FRACTION = 0.42

STATUS_OK, STATUS_BACKGROUND, STATUS_BAD_INPUT, STATUS_SOLVE_FAILED = 0, 1, 2, 3


# ----------------------------------------------------------------------------------------------
# parameters (mirror of apic_params in include/apic.h; independent definition)
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass
class OracleParams:
    tile_n: int
    upsample: int
    wavelength_um: float
    pixel_um: float
    na_obj: float
    k_bright: np.ndarray                   # [n_bright][2] cycles/um
    k_dark: np.ndarray                     # [n_dark][2]
    noll: Sequence[int]                    # fitted Noll indices, each >= 4 (R9)
    kk_pad: int = 1
    refine_iters: int = 3
    intensity_floor: float = 1e-6
    bg_mode: int = 0
    bg_threshold: float = 0.0
    dark_order: str = "sequential"         # R15 "sequential" (the contract) | "ring" (second reading R15b)

    @property
    def radius(self) -> float:
        return self.na_obj * self.tile_n * self.pixel_um / self.wavelength_um

    @property
    def kappa_bright(self) -> np.ndarray:
        return np.asarray(self.k_bright, dtype=np.float64).reshape(-1, 2) * (self.tile_n * self.pixel_um)

    @property
    def kappa_dark(self) -> np.ndarray:
        if self.k_dark is None or len(self.k_dark) == 0:
            return np.zeros((0, 2))
        return np.asarray(self.k_dark, dtype=np.float64).reshape(-1, 2) * (self.tile_n * self.pixel_um)


# ----------------------------------------------------------------------------------------------
# O0: transforms and grids
# ----------------------------------------------------------------------------------------------
def signed_bins(n: int) -> np.ndarray:
    """Signed integer bins in FFT order (0..n/2-1, -n/2..-1)."""
    k = np.arange(n)
    return np.where(k < n // 2, k, k - n).astype(np.int64)


def fft2n(a: np.ndarray) -> np.ndarray:
    """Normalised forward transform: S[k] = (1/N^2) sum_x s[x] e^{-j2pi k.x/N}  (O0)."""
    return np.fft.fft2(a) / float(a.shape[-1] * a.shape[-2])


def ifft2u(spec: np.ndarray) -> np.ndarray:
    """Unscaled inverse: s[x] = sum_k S[k] e^{+j2pi k.x/N} (inverse of fft2n)."""
    return np.fft.ifft2(spec) * float(spec.shape[-1] * spec.shape[-2])


def naive_dft2(a: np.ndarray, inverse: bool = False) -> np.ndarray:
    """The definition of the 2-D DFT as two dense matrix products, O(N^3) work per axis pair
    (N <= 128).  Unnormalised: forward sign -, inverse sign + (no 1/N^2)."""
    n0, n1 = a.shape
    sgn = +1.0 if inverse else -1.0
    w0 = np.exp(sgn * 1j * TWO_PI * np.outer(np.arange(n0), np.arange(n0)) / n0)
    w1 = np.exp(sgn * 1j * TWO_PI * np.outer(np.arange(n1), np.arange(n1)) / n1)
    return w0 @ a @ w1.T


# ----------------------------------------------------------------------------------------------
# Zernike polynomials, Noll ordering and normalisation (R9; BASELINE.json item 3)
# ----------------------------------------------------------------------------------------------
def noll_to_nm(j: int) -> Tuple[int, int]:
    """Noll index j >= 1 -> (n, m); m > 0 cosine (even j), m < 0 sine (odd j)."""
    if j < 1:
        raise ValueError("Noll index starts at 1")
    n = int(math.ceil((-3.0 + math.sqrt(9.0 + 8.0 * (j - 1))) / 2.0))
    first = n * (n + 1) // 2 + 1                 # first j of radial order n
    pos = j - first                              # 0..n within the order
    if n % 2 == 0:
        am = 2 * ((pos + 1) // 2)
    else:
        am = 2 * (pos // 2) + 1
    if am == 0:
        return n, 0
    return n, (am if j % 2 == 0 else -am)


def zernike_radial(n: int, am: int, rho: np.ndarray) -> np.ndarray:
    """R_n^{|m|}(rho) = sum_s (-1)^s (n-s)! / (s! ((n+m)/2-s)! ((n-m)/2-s)!) rho^(n-2s)."""
    out = np.zeros_like(rho, dtype=np.float64)
    for s in range((n - am) // 2 + 1):
        c = ((-1) ** s) * math.factorial(n - s) / (
            math.factorial(s) * math.factorial((n + am) // 2 - s) * math.factorial((n - am) // 2 - s))
        out = out + c * rho ** (n - 2 * s)
    return out


def zernike(j: int, rho: np.ndarray, theta: np.ndarray) -> np.ndarray:
    """Z_j(rho, theta), unit RMS over the unit disc (Noll 1976).  Evaluated as a polynomial
    also where rho marginally exceeds 1 (O0)."""
    n, m = noll_to_nm(j)
    am = abs(m)
    rad = zernike_radial(n, am, rho)
    if m == 0:
        return math.sqrt(n + 1.0) * rad
    if m > 0:
        return math.sqrt(2.0 * (n + 1.0)) * rad * np.cos(am * theta)
    return math.sqrt(2.0 * (n + 1.0)) * rad * np.sin(am * theta)


def zernike_at_bins(j: int, kx: np.ndarray, ky: np.ndarray, kappa: Sequence[float], radius: float) -> np.ndarray:
    """Z_j at pupil coordinate (k + kappa)/R  (the pupil is sampled off-lattice, R2)."""
    px = (np.asarray(kx, dtype=np.float64) + kappa[0]) / radius
    py = (np.asarray(ky, dtype=np.float64) + kappa[1]) / radius
    return zernike(j, np.hypot(px, py), np.arctan2(py, px))


def pupil_phase(noll: Sequence[int], coef: Sequence[float], kx, ky, kappa, radius) -> np.ndarray:
    """phi_hat(k + kappa) = sum_j c_j Z_j((k + kappa)/R)."""
    kx = np.asarray(kx)
    ky = np.asarray(ky)
    out = np.zeros(np.broadcast(kx, ky).shape)
    for j, c in zip(noll, coef):
        out = out + c * zernike_at_bins(j, kx, ky, kappa, radius)
    return out


# ----------------------------------------------------------------------------------------------
# geometry that depends only on (N, R, kappa): discs, pair overlaps, darkfield index sets
# ----------------------------------------------------------------------------------------------
class Geometry:
    """All index sets of the path on the centred grid: arrays are [N][N] with element
    [iy][ix] <-> bin (kx, ky) = (ix - N/2, iy - N/2)."""

    def __init__(self, p: OracleParams):
        self.p = p
        n = p.tile_n
        self.n = n
        self.radius = p.radius
        c = np.arange(n) - n // 2
        self.kx, self.ky = np.meshgrid(c, c, indexing="xy")        # centred
        self.kappa_b = p.kappa_bright
        self.kappa_d = p.kappa_dark
        self.disc_b = [self.disc(k) for k in self.kappa_b]
        self.disc_d = [self.disc(k) for k in self.kappa_d]
        # R3: the DC bin lies inside every NA-matching disc
        for i, m in enumerate(self.disc_b):
            if not m[n // 2, n // 2]:
                raise ValueError(f"NA-matching LED {i}: DC bin is outside its disc")
        self.pairs = self._pairs()
        self.dark_order = self._dark_order()

    def disc(self, kappa) -> np.ndarray:
        """D_i = {k : |k + kappa_i|^2 <= R^2 (1 + 1e-9)}  (Eq. 7 support; R3)."""
        return ((self.kx + kappa[0]) ** 2 + (self.ky + kappa[1]) ** 2) <= self.radius ** 2 * (1.0 + DISC_RTOL)

    def _pairs(self) -> List[Tuple[int, int]]:
        """All i<l with |D_i ∩ D_l| >= 2 (Eq. 8; R12)."""
        out = []
        for i, l in itertools.combinations(range(len(self.disc_b)), 2):
            if np.count_nonzero(self.disc_b[i] & self.disc_b[l]) >= 2:
                out.append((i, l))
        return out

    def _dark_order(self) -> List[int]:
        """R15: ascending |kappa| (rounded to 1e-6 bins), ties by input order."""
        key = [(int(round(float(np.hypot(*k)) / KAPPA_ORDER_QUANTUM)), i) for i, k in enumerate(self.kappa_d)]
        return [i for _, i in sorted(key)]

    def _dark_rings(self) -> List[List[int]]:
        """Darkfield LEDs grouped by |kappa| (same rounding as the order), rings in ascending |kappa|."""
        rings: Dict[int, List[int]] = {}
        for i in self._dark_order():
            rings.setdefault(int(round(float(np.hypot(*self.kappa_d[i])) / KAPPA_ORDER_QUANTUM)), []).append(i)
        return [rings[k] for k in sorted(rings)]

    def to_centred(self, a_fft_order: np.ndarray) -> np.ndarray:
        return np.fft.fftshift(a_fft_order, axes=(-2, -1))

    def to_fft_order(self, a_centred: np.ndarray) -> np.ndarray:
        return np.fft.ifftshift(a_centred, axes=(-2, -1))


def minkowski_difference(a_mask: np.ndarray, b_mask: np.ndarray) -> np.ndarray:
    """{a - b : a in A, b in B} as a centred boolean grid of the same size.  Written out as the
    definition (all pairs); supports never wrap (R16), which is asserted."""
    n = a_mask.shape[0]
    ay, ax = np.nonzero(a_mask)
    by, bx = np.nonzero(b_mask)
    out = np.zeros_like(a_mask, dtype=bool)
    if ay.size == 0 or by.size == 0:
        return out
    # process in chunks of A to bound memory
    chunk = max(1, int(4_000_000 // max(1, by.size)))
    for s in range(0, ay.size, chunk):
        dy = (ay[s:s + chunk, None] - by[None, :]).ravel()
        dx = (ax[s:s + chunk, None] - bx[None, :]).ravel()
        if (np.abs(dy).max() >= n // 2) or (np.abs(dx).max() >= n // 2):
            raise ValueError("index-set difference would wrap around the grid")
        out[dy + n // 2, dx + n // 2] = True
    return out


@dataclasses.dataclass
class DarkSets:
    led: int                 # index into the darkfield list (input order)
    P: np.ndarray            # centred bool: D_i ∩ known
    U: np.ndarray            # centred bool: D_i \ known
    Q: np.ndarray            # centred bool: linear region
    unknown_fraction: float
    ring: int = 0            # index of the LED's ring (equal |kappa|), ascending


def darkfield_sets(geo: Geometry) -> Tuple[List[DarkSets], np.ndarray]:
    """O6 index sets for every darkfield LED in processing order (Eq. 13 region Q_i,
    PAPER.md:130-132; R15, R16).  Returns (list, final known mask).

    PAPER.md:135 extends the spectrum "across all darkfield measurements" without stating an order.
    R15 (``dark_order = "sequential"``, the contract): one LED after the other, ``known`` grows after
    every LED, a bin belongs to the first LED that solves it.  R15b (``"ring"``): every LED of a ring
    (equal |kappa|) is solved against ``known`` as it stands when the ring starts; ``known`` grows once
    per ring (bins solved by several LEDs of the ring are averaged in darkfield_extend)."""
    known = np.zeros((geo.n, geo.n), dtype=bool)
    for m in geo.disc_b:
        known |= m
    ring_wise = geo.p.dark_order == "ring"
    if geo.p.dark_order not in ("sequential", "ring"):
        raise ValueError("dark_order must be 'sequential' or 'ring'")
    out: List[DarkSets] = []
    for ri, ring in enumerate(geo._dark_rings()):
        start = known.copy()
        for led in ring:
            base = start if ring_wise else known
            d = geo.disc_d[led]
            P = d & base
            U = d & ~base
            if not U.any():
                continue
            known = _dark_sets_one(out, led, ri, d, P, U, known)
    return out, known


def _dark_sets_one(out, led, ring, d, P, U, known):
    """Checks and the linear region Q of one LED (Eq. 13; R16); appends to ``out`` and returns known ∪ U."""
    frac = U.sum() / float(d.sum())
    if frac > MAX_UNKNOWN_FRACTION:
        raise ValueError(f"darkfield LED {led}: unknown fraction {frac:.3f} > 0.42 (PAPER.md:201)")
    cross = minkowski_difference(U, P)          # supp(U ⋆ P) = {u - p}
    other = minkowski_difference(P, U)          # supp(P ⋆ U) = {p - u}
    auto = minkowski_difference(U, U)           # supp(U ⋆ U) = {u - u'}
    Q = cross & ~(other | auto)
    if not Q.any():
        raise ValueError(f"darkfield LED {led}: empty linear region Q")
    out.append(DarkSets(led=led, P=P, U=U, Q=Q, unknown_fraction=frac, ring=ring))
    return known | U


# ----------------------------------------------------------------------------------------------
# O1: background flag (PAPER.md:179 uses a variance threshold; BASELINE.json item 5 a mean one; R18)
# ----------------------------------------------------------------------------------------------
def background_flag(stack_bright: np.ndarray, bg_mode: int, bg_threshold: float) -> bool:
    if bg_mode == 0:
        return False
    x = np.asarray(stack_bright, dtype=np.float64)
    mean = x.mean()
    if bg_mode == 1:
        return bool(mean >= bg_threshold)
    if bg_mode == 2:
        return bool(x.var() / (mean * mean) <= bg_threshold)
    raise ValueError("bg_mode")


# ----------------------------------------------------------------------------------------------
# O2: Kramers-Kronig field retrieval (Eq. 4-6; R4-R7)
# ----------------------------------------------------------------------------------------------
def halfplane_weight(n: int, kappa: Sequence[float]) -> np.ndarray:
    """w(k) of Eq. 5 in FFT order: 1 where k.kappa<0, 1/2 on the line, 0 where >0;
    tolerance tau on the normalised dot product; sign-less Nyquist rows/columns get 1/2 (R5)."""
    k = signed_bins(n).astype(np.float64)
    kap = np.asarray(kappa, dtype=np.float64)
    d = (k[None, :] * kap[0] + k[:, None] * kap[1]) / math.hypot(kap[0], kap[1])
    w = np.where(d < -HALFPLANE_TAU, 1.0, np.where(d > HALFPLANE_TAU, 0.0, 0.5))
    nyq = (k == -(n // 2))
    w[nyq, :] = 0.5
    w[:, nyq] = 0.5
    return w


def fourier_resample(a: np.ndarray, m: int) -> np.ndarray:
    """Band-limited resampling of an N x N array to m x m (m > N zero-pads the spectrum, m < N
    crops it); the N/2 Nyquist bin is split evenly when padding.  Values at common points are
    preserved (no extra scaling)."""
    n = a.shape[0]
    spec = np.fft.fftshift(fft2n(a))
    out = np.zeros((m, m), dtype=np.complex128)
    if m >= n:
        o = m // 2 - n // 2
        out[o:o + n, o:o + n] = spec
        if m > n:                              # split the sign-less Nyquist row/column
            out[o, :] *= 0.5
            out[o + n, :] = out[o, :]
            out[:, o] *= 0.5
            out[:, o + n] = out[:, o]
    else:
        o = n // 2 - m // 2
        out[:, :] = spec[o:o + m, o:o + m]
    return ifft2u(np.fft.ifftshift(out))


def kk_field(intensity: np.ndarray, kappa: Sequence[float], floor: float = 1e-6, pad: int = 1) -> np.ndarray:
    """s_i(x) = S'_i(x) e^{-j theta_i} = exp(F^{-1}[w ⊙ F(log I_i)])   (Eq. 5-6).

    R6: I <- max(I, floor*mean(I)).  R7: with pad>1 the intensity is first Fourier-interpolated
    to the pad*N grid and the recovered field is band-limited back to N afterwards.
    """
    img = np.asarray(intensity, dtype=np.float64)
    n = img.shape[0]
    if pad > 1:
        img = fourier_resample(img, pad * n).real
    img = np.maximum(img, floor * img.mean())
    big = np.fft.fft2(np.log(img))
    w = halfplane_weight(img.shape[0], kappa)
    s = np.exp(np.fft.ifft2(w * big))
    if pad > 1:
        s = fourier_resample(s, n)
    return s


def sub_spectrum(s: np.ndarray) -> np.ndarray:
    """O3: S_hat_i = F(s_i)/N^2 (Eq. 7), full grid, FFT order."""
    return fft2n(s)


# ----------------------------------------------------------------------------------------------
# O4: aberration extraction (Eq. 8-10; R8-R12)
# ----------------------------------------------------------------------------------------------
def aberration_rows(geo: Geometry, i: int, l: int):
    """For pair (i, l): overlap bins K in S_il and rows
    a_j(K) = Z_j(K+kappa_i) - Z_j(K+kappa_l) - Z_j(kappa_i) + Z_j(kappa_l)   (Eq. 10 with R8).
    Returns (mask [N][N] centred, iy, ix, A [rows][n_z])."""
    p = geo.p
    mask = geo.disc_b[i] & geo.disc_b[l]
    iy, ix = np.nonzero(mask)
    kx = geo.kx[iy, ix]
    ky = geo.ky[iy, ix]
    zero = np.zeros(1)
    cols = []
    for j in p.noll:
        a = (zernike_at_bins(j, kx, ky, geo.kappa_b[i], geo.radius)
             - zernike_at_bins(j, kx, ky, geo.kappa_b[l], geo.radius)
             - zernike_at_bins(j, zero, zero, geo.kappa_b[i], geo.radius)[0]
             + zernike_at_bins(j, zero, zero, geo.kappa_b[l], geo.radius)[0])
        cols.append(a)
    return mask, iy, ix, np.stack(cols, axis=1) if cols else np.zeros((iy.size, 0))


def wrap_phase(x: np.ndarray) -> np.ndarray:
    """wrap(x) = x - 2 pi round(x / 2 pi)   (R11)."""
    return x - TWO_PI * np.round(x / TWO_PI)


def weighted_solve(a: np.ndarray, b: np.ndarray, w: np.ndarray) -> np.ndarray:
    """argmin_c sum_r w_r (a_r.c - b_r)^2 via the normal equations (A^T W A) c = A^T W b."""
    aw = a * w[:, None]
    return np.linalg.solve(a.T @ aw, aw.T @ b)


def solve_aberration(geo: Geometry, spectra_centred: Sequence[np.ndarray], refine_iters: int,
                     c_init: Optional[np.ndarray] = None):
    """O4.  spectra_centred[i] = S_hat_i on the centred grid (only D_i is read).
    Returns (c [n_z], status, info dict with row counts / residual).
    c_init (reading B9: "initialise S6 from neighbours"; the paper shows the pupil
    varying smoothly over the slide, Fig. 4(b)): a prior for the coefficients, e.g. the slide-level fit
    of pupil_field_fit evaluated at this tile.  It REPLACES the gradient-domain start c^0; the re-wrapped refinement
    steps and the status rule are unchanged, so inside the basin of R11 the result is the same minimiser."""
    full_a, full_beta, full_w = [], [], []
    grad_a, grad_b, grad_w = [], [], []
    for (i, l) in geo.pairs:
        mask, iy, ix, a = aberration_rows(geo, i, l)
        prod = spectra_centred[i][iy, ix] * np.conj(spectra_centred[l][iy, ix])    # Eq. 9
        full_a.append(a)
        full_beta.append(np.angle(prod))
        full_w.append(np.abs(prod))                                               # R10
        # (i) gradient rows: K and K+e both in S_il, e in {x, y}
        row_of = -np.ones(mask.shape, dtype=np.int64)
        row_of[iy, ix] = np.arange(iy.size)
        for (dy, dx) in ((0, 1), (1, 0)):
            y2, x2 = iy + dy, ix + dx
            ok = (y2 < geo.n) & (x2 < geo.n)
            ok[ok] &= mask[y2[ok], x2[ok]]
            r0 = np.nonzero(ok)[0]
            r1 = row_of[y2[ok], x2[ok]]
            grad_a.append(a[r1] - a[r0])
            grad_b.append(np.angle(prod[r1] * np.conj(prod[r0])))
            grad_w.append(np.abs(prod[r1]) * np.abs(prod[r0]))
    a_full = np.concatenate(full_a)
    beta = np.concatenate(full_beta)
    w_full = np.concatenate(full_w)
    a_grad = np.concatenate(grad_a)
    if c_init is None:
        c = weighted_solve(a_grad, np.concatenate(grad_b), np.concatenate(grad_w))  # c^0
    else:
        c = np.asarray(c_init, dtype=np.float64).copy()                              # B9
    normal = a_full.T @ (a_full * w_full[:, None])
    for _ in range(refine_iters):                                                  # (ii)
        r = wrap_phase(beta - a_full @ c)
        c = c + np.linalg.solve(normal, a_full.T @ (w_full * r))
    r = wrap_phase(beta - a_full @ c)
    rms = math.sqrt(float((w_full * r * r).sum() / w_full.sum()))
    status = STATUS_SOLVE_FAILED if (not np.isfinite(rms) or rms > 1.0) else STATUS_OK
    info = dict(rows=a_full.shape[0], grad_rows=a_grad.shape[0], pairs=len(geo.pairs),
                residual_rms=rms, cond=float(np.linalg.cond(normal)))
    return c, status, info


# ----------------------------------------------------------------------------------------------
# O5: correction + stitching (R13, R14)
# ----------------------------------------------------------------------------------------------
def stitch(geo: Geometry, spectra_centred: Sequence[np.ndarray], coef: np.ndarray):
    """O_hat(k) = mean over {i: k in D_i} of S_hat_i(k) exp(-j[phi_hat(k+kappa_i) - phi_hat(kappa_i)]).
    Returns (O_hat centred [N][N], known mask)."""
    p = geo.p
    acc = np.zeros((geo.n, geo.n), dtype=np.complex128)
    cnt = np.zeros((geo.n, geo.n), dtype=np.int64)
    zero = np.zeros(1)
    for i, mask in enumerate(geo.disc_b):
        iy, ix = np.nonzero(mask)
        phi = pupil_phase(p.noll, coef, geo.kx[iy, ix], geo.ky[iy, ix], geo.kappa_b[i], geo.radius)
        theta = pupil_phase(p.noll, coef, zero, zero, geo.kappa_b[i], geo.radius)[0]
        acc[iy, ix] += spectra_centred[i][iy, ix] * np.exp(-1j * (phi - theta))
        cnt[iy, ix] += 1
    known = cnt > 0
    out = np.zeros_like(acc)
    out[known] = acc[known] / cnt[known]
    return out, known


# ----------------------------------------------------------------------------------------------
# O6: darkfield extension (Eq. 11-13; R15-R17)
# ----------------------------------------------------------------------------------------------
def correlate_fft(a_centred: np.ndarray, b_centred: np.ndarray) -> np.ndarray:
    """[A ⋆ B](k) = sum_q A(q+k) conj B(q) (circular on the N grid), centred in / centred out."""
    a = ifft2u(np.fft.ifftshift(a_centred))
    b = ifft2u(np.fft.ifftshift(b_centred))
    return np.fft.fftshift(fft2n(a * np.conj(b)))


def correlate_direct(a_centred: np.ndarray, b_centred: np.ndarray, at_mask: np.ndarray) -> np.ndarray:
    """The same correlation as an explicit double sum, evaluated on ``at_mask`` only (pin for
    correlate_fft; small cases)."""
    n = a_centred.shape[0]
    out = np.zeros_like(a_centred, dtype=np.complex128)
    by, bx = np.nonzero(b_centred)
    for ky, kx in zip(*np.nonzero(at_mask)):
        y = by + (ky - n // 2)
        x = bx + (kx - n // 2)
        ok = (y >= 0) & (y < n) & (x >= 0) & (x < n)
        out[ky, kx] = np.sum(a_centred[y[ok], x[ok]] * np.conj(b_centred[by[ok], bx[ok]]))
    return out


def darkfield_matrix(p_hat: np.ndarray, P: np.ndarray, U: np.ndarray, Q: np.ndarray) -> np.ndarray:
    """C[k, u] = conj P_hat(u - k) for k in Q, u in U (0 where u-k is outside P)  - the
    block-Toeplitz matrix of PAPER.md:135.  Row/column order = row-major order of the masks."""
    n = p_hat.shape[0]
    qy, qx = np.nonzero(Q)
    uy, ux = np.nonzero(U)
    dy = uy[None, :] - (qy[:, None] - n // 2)       # index of bin (u - k) on the centred grid
    dx = ux[None, :] - (qx[:, None] - n // 2)
    ok = (dy >= 0) & (dy < n) & (dx >= 0) & (dx < n)
    dyc = np.where(ok, dy, 0)
    dxc = np.where(ok, dx, 0)
    vals = np.conj(p_hat[dyc, dxc])
    vals[~(ok & P[dyc, dxc])] = 0.0
    return vals


def darkfield_extend(geo: Geometry, o_hat: np.ndarray, known: np.ndarray, coef: np.ndarray,
                     dark_stack: np.ndarray, sets: Optional[List[DarkSets]] = None,
                     collect: Optional[list] = None):
    """O6: for each darkfield LED in order, solve C U_hat = F(I)/N^2 - P_hat⋆P_hat on Q in the
    least-squares sense and extend the object spectrum.  Returns (O_hat, known)."""
    p = geo.p
    if sets is None:
        sets, _ = darkfield_sets(geo)
    o_hat = o_hat.copy()
    known = known.copy()
    ring_wise = p.dark_order == "ring"
    for ri in sorted({ds.ring for ds in sets}):
        ring = [ds for ds in sets if ds.ring == ri]
        # R15b: every LED of the ring reads the spectrum and the known set as they stand when the ring starts;
        # a bin solved by several LEDs of the ring gets the unweighted mean of their solutions (the rule of R13)
        o_start, known_start = o_hat.copy(), known.copy()
        acc = np.zeros_like(o_hat)
        cnt = np.zeros(o_hat.shape, dtype=np.int64)
        for ds in ring:
            o_src, k_src = (o_start, known_start) if ring_wise else (o_hat, known)
            kap = geo.kappa_d[ds.led]
            if not np.array_equal(ds.P, geo.disc_d[ds.led] & k_src):
                raise AssertionError("darkfield index sets out of sync with the known region")
            phi = pupil_phase(p.noll, coef, geo.kx, geo.ky, kap, geo.radius)
            p_hat = np.where(ds.P, o_src * np.exp(1j * phi), 0.0)
            spec_i = np.fft.fftshift(fft2n(np.asarray(dark_stack[ds.led], dtype=np.float64)))
            rhs_grid = spec_i - correlate_fft(p_hat, p_hat)                   # Eq. 13 lhs
            d = rhs_grid[ds.Q]
            cmat = darkfield_matrix(p_hat, ds.P, ds.U, ds.Q)
            u_hat, *_ = np.linalg.lstsq(cmat, d, rcond=None)
            if ring_wise:
                acc[ds.U] += u_hat * np.exp(-1j * phi[ds.U])
                cnt[ds.U] += 1
            else:
                o_hat[ds.U] = u_hat * np.exp(-1j * phi[ds.U])
                known = known | ds.U
            if collect is not None:
                collect.append(dict(led=ds.led, u_hat=u_hat, d=d, p_hat=p_hat,
                                    resid=float(np.linalg.norm(cmat @ u_hat - d) / max(np.linalg.norm(d), 1e-300))))
        if ring_wise:
            solved = cnt > 0
            o_hat[solved] = acc[solved] / cnt[solved]
            known = known | solved
    return o_hat, known


# ----------------------------------------------------------------------------------------------
# O7: outputs
# ----------------------------------------------------------------------------------------------
def output_field(o_hat_centred: np.ndarray, upsample: int) -> np.ndarray:
    """f[X] = sum_k O_hat(k) e^{+j 2 pi k.X/(uN)}, X in [0,uN)^2: zero-padded inverse DFT with no
    extra scaling (a blank object gives f = 1)."""
    n = o_hat_centred.shape[0]
    m = n * upsample
    big = np.zeros((m, m), dtype=np.complex128)
    o = m // 2 - n // 2
    big[o:o + n, o:o + n] = o_hat_centred
    return ifft2u(np.fft.ifftshift(big))


def pupil_function(geo: Geometry, coef: np.ndarray) -> np.ndarray:
    """1[|k|<=R] e^{j phi_hat(k)} on the centred N x N grid (bin 0 at index N/2)."""
    mask = geo.disc((0.0, 0.0))
    phi = pupil_phase(geo.p.noll, coef, geo.kx, geo.ky, (0.0, 0.0), geo.radius)
    return np.where(mask, np.exp(1j * phi), 0.0)


@dataclasses.dataclass
class OracleResult:
    status: int
    field: np.ndarray                    # [uN][uN] complex128
    zernike: np.ndarray                  # [n_z] rad
    pupil: np.ndarray                    # [N][N] complex128, centred
    o_hat: Optional[np.ndarray] = None   # centred object spectrum
    known: Optional[np.ndarray] = None
    spectra: Optional[List[np.ndarray]] = None   # centred S_hat_i (full grid)
    info: Optional[dict] = None


def reconstruct_tile(stack: np.ndarray, p: OracleParams, geo: Optional[Geometry] = None,
                     sets: Optional[List[DarkSets]] = None, keep: bool = False,
                     zernike_init: Optional[np.ndarray] = None) -> OracleResult:
    """The whole hot path O1..O7 for one tile.  stack: [n_bright+n_dark][N][N]."""
    n = p.tile_n
    nb = len(p.k_bright)
    nz = len(p.noll)
    geo = geo or Geometry(p)
    x = np.asarray(stack)
    zeros = OracleResult(status=STATUS_OK, field=np.zeros((n * p.upsample,) * 2, complex),
                         zernike=np.zeros(nz), pupil=np.zeros((n, n), complex))
    if not np.all(np.isfinite(x)):
        zeros.status = STATUS_BAD_INPUT
        return zeros
    if background_flag(x[:nb], p.bg_mode, p.bg_threshold):                   # O1
        zeros.status = STATUS_BACKGROUND
        return zeros
    spectra = []
    for i in range(nb):                                                       # O2, O3
        s = kk_field(x[i], geo.kappa_b[i], floor=p.intensity_floor, pad=p.kk_pad)
        spectra.append(np.where(geo.disc_b[i], np.fft.fftshift(sub_spectrum(s)), 0.0))
    coef, status, info = solve_aberration(geo, spectra, p.refine_iters, c_init=zernike_init)   # O4 (B9)
    o_hat, known = stitch(geo, spectra, coef)                                 # O5
    if len(p.k_dark):
        o_hat, known = darkfield_extend(geo, o_hat, known, coef, x[nb:], sets=sets)   # O6
    res = OracleResult(status=status, field=output_field(o_hat, p.upsample), zernike=coef,
                       pupil=pupil_function(geo, coef), info=info)
    if keep:
        res.o_hat, res.known, res.spectra = o_hat, known, spectra
    return res


def reconstruct_batch(stacks: np.ndarray, p: OracleParams) -> List[OracleResult]:
    geo = Geometry(p)
    sets = darkfield_sets(geo)[0] if len(p.k_dark) else None
    return [reconstruct_tile(s, p, geo=geo, sets=sets) for s in stacks]
