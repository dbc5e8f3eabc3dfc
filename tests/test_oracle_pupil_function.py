"""Pins for the oracle's third output, O7 `pupil_function`: P(k) = 1[|k| <= R] e^{+j phi_hat(k)} on the centred
N x N grid (Eq. 2: the coherent transfer function is the pupil disc times e^{j phi}; the
recovered aberration is returned with the object).  Three things a slip would break: the support and its centring
(bin 0 at index N/2), the radial profile (defocus closed form at named bins), and the sign of the exponent (equality
with the generator's own forward-model CTF, which builds its Zernikes through a different formula)."""
import math

import numpy as np
import pytest

from apic_synth import get_config
from apic_synth.forward import pupil_phase_at
from oracle import apic_oracle as O
from helpers import oracle_params


@pytest.mark.parametrize("idx", [0, 2])
def test_zero_coefficients_give_the_disc_centred_on_bin_zero(idx):
    cfg = get_config(idx)
    geo = O.Geometry(oracle_params(cfg))
    n, r = cfg.tile_n, cfg.pupil_radius_bins
    p = O.pupil_function(geo, np.zeros(len(cfg.noll_fit)))
    assert p.shape == (n, n)
    k = np.arange(n) - n // 2                                   # bin index of array index i is i - N/2
    inside = (k[None, :] ** 2 + k[:, None] ** 2) <= r * r * (1 + 1e-9)
    assert np.array_equal(p != 0, inside)                       # exactly the bins with |k| <= R
    assert np.all(p[inside] == 1.0)
    assert p[n // 2, n // 2] == 1.0 and p[0, 0] == 0.0
    # the disc is symmetric about index N/2, not about (N-1)/2: row N/2 + m equals row N/2 - m
    m = int(r)
    assert p[n // 2 + m, n // 2] == 1.0 and p[n // 2 - m, n // 2] == 1.0 and p[n // 2 - m - 1, n // 2] == 0.0
    assert np.count_nonzero(p) == np.count_nonzero(geo.disc((0.0, 0.0)))


def test_pure_defocus_has_the_closed_form_phase_at_named_bins():
    cfg = get_config(2)
    geo = O.Geometry(oracle_params(cfg))
    n, r = cfg.tile_n, cfg.pupil_radius_bins
    j4 = list(cfg.noll_fit).index(4)
    c = np.zeros(len(cfg.noll_fit))
    c[j4] = 0.37
    p = O.pupil_function(geo, c)
    for kx, ky in [(0, 0), (10, 0), (0, -17), (-20, 21), (int(r), 0)]:
        want = 0.37 * math.sqrt(3.0) * (2.0 * (kx * kx + ky * ky) / (r * r) - 1.0)   # Z4 = sqrt(3) (2 rho^2 - 1)
        got = p[n // 2 + ky, n // 2 + kx]                                           # row = ky, column = kx
        assert abs(abs(got) - 1.0) < 1e-14
        assert abs(np.angle(got * np.exp(-1j * want))) < 1e-12


def test_astigmatism_orientation_and_exponent_sign_match_the_forward_model():
    """The generator images through mask * e^{+j phi} (apic_synth/forward.py); the oracle's pupil with the same
    coefficients must be that CTF, bin for bin - a conjugated exponent, swapped axes or a shifted centre all fail."""
    cfg = get_config(2)
    geo = O.Geometry(oracle_params(cfg))
    rng = np.random.default_rng(3)
    c = rng.normal(0.0, 0.4, len(cfg.noll_fit))
    mask, phi = pupil_phase_at(cfg, {j: v for j, v in zip(cfg.noll_fit, c)}, np.zeros(2))
    ctf = np.fft.fftshift(np.where(mask, np.exp(1j * phi), 0.0))
    p = O.pupil_function(geo, c)
    assert np.array_equal(p != 0, ctf != 0)
    assert np.abs(p - ctf).max() < 1e-12
    assert np.abs(p - np.conj(ctf)).max() > 0.5                 # the check can tell the two signs apart
    assert np.abs(p - ctf.T).max() > 0.5                        # ... and the two axes
