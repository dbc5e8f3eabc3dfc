"""Pins for the forward model (generator) and the Kramers-Kronig step (Eq. 4-7)."""
import dataclasses

import numpy as np
import pytest

from apic_synth import get_config, led_kvectors, make_tile
from apic_synth.forward import forward_stack, object_spectrum_raw, pupil_phase_at
from oracle import apic_oracle as O
from helpers import oracle_params, rel_l2


def _true_field(cfg, truth, kappa):
    """S'_i(x) of the forward model (generator side), fp64."""
    mask, phi = pupil_phase_at(cfg, truth.coef, kappa)
    s_hat = np.where(mask, object_spectrum_raw(cfg, truth.obj) * np.exp(1j * phi), 0.0)
    return np.fft.ifft2(s_hat) * cfg.tile_n ** 2, s_hat


def test_blank_object_gives_unit_brightfield_and_zero_darkfield():
    cfg = get_config(2, tile_n=64, batch=1, grid=(1, 1))
    stack, truth = make_tile(cfg, 0, noise="none", blank=True, keep_clean=True)
    assert np.abs(truth.clean[:cfg.n_bright] - 1.0).max() < 1e-12
    assert np.abs(truth.clean[cfg.n_bright:]).max() < 1e-20


def test_intensity_spectrum_is_bandlimited_to_2R():
    cfg = get_config(0)
    _, truth = make_tile(cfg, 0, keep_clean=True)
    p = oracle_params(cfg)
    geo = O.Geometry(p)
    for img in truth.clean:
        spec = np.fft.fftshift(O.fft2n(img))
        outside = (geo.kx ** 2 + geo.ky ** 2) > (2 * geo.radius) ** 2 * (1 + 1e-9)
        assert np.abs(spec[outside]).max() < 1e-13 * np.abs(spec).max()


def test_na_matching_condition_on_lattice():
    # every in-disc bin except DC lies strictly in the half plane k.kappa < 0
    for idx in (0, 1):
        cfg = get_config(idx)
        geo = O.Geometry(oracle_params(cfg))
        for kap, mask in zip(geo.kappa_b, geo.disc_b):
            d = geo.kx * kap[0] + geo.ky * kap[1]
            inside = mask.copy()
            inside[cfg.tile_n // 2, cfg.tile_n // 2] = False
            assert d[inside].max() < -O.HALFPLANE_TAU * np.hypot(*kap)


def test_halfplane_weight_special_values():
    n = 64
    w = O.halfplane_weight(n, (10.0, 0.0))           # azimuth 0: whole kx=0 column is "on the line"
    k = O.signed_bins(n)
    assert np.all(w[:, k == 0] == 0.5)
    assert np.all(w[:, k == -n // 2] == 0.5) and np.all(w[k == -n // 2, :] == 0.5)
    inner = (k != -n // 2)
    assert np.all(w[np.ix_(inner, (k < 0) & inner)] == 1.0)
    assert np.all(w[np.ix_(inner, k > 0)] == 0.0)
    # w(k) + w(-k) = 1 everywhere: the masked spectrum's Hermitian part is L/2, so Re g = (log I)/2
    w2 = O.halfplane_weight(n, (3.3, -7.1))
    idx = (-np.arange(n)) % n
    assert np.allclose(w2 + w2[np.ix_(idx, idx)], 1.0)


@pytest.mark.parametrize("led", [0, 1, 2, 3])
def test_kk_is_exact_and_error_decays_with_padding(led):
    """Exact result: KK recovers S'_i e^{-j arg DC}; the only error is aliasing of the harmonics
    of log I, which decays with Fourier pre-upsampling (2e-4 -> <=4e-9 -> <=3e-16)."""
    cfg = get_config(0)
    _, truth = make_tile(cfg, 0, keep_clean=True)
    p = oracle_params(cfg)
    kap = p.kappa_bright[led]
    field, s_hat = _true_field(cfg, truth, kap)
    target = field * np.exp(-1j * np.angle(s_hat[0, 0]))
    errs = [rel_l2(O.kk_field(truth.clean[led], kap, pad=pad), target) for pad in (1, 2, 4)]
    assert errs[0] < 2e-3
    assert errs[1] < 1e-7 and errs[1] < errs[0] * 1e-3
    assert errs[2] < 1e-12


def test_kk_modulus_dc_and_support():
    cfg = get_config(0)
    _, truth = make_tile(cfg, 0, keep_clean=True)
    p = oracle_params(cfg)
    geo = O.Geometry(p)
    for led in range(cfg.n_bright):
        s = O.kk_field(truth.clean[led], p.kappa_bright[led], pad=1)
        assert np.abs(np.abs(s) ** 2 - truth.clean[led]).max() < 1e-12       # |s|^2 = I pointwise
        spec = O.sub_spectrum(s)
        # DC real-positive (R14), up to the pad-1 aliasing floor
        assert abs(spec[0, 0].imag) < 1e-6 * abs(spec[0, 0]) and spec[0, 0].real > 0
        c = np.fft.fftshift(spec)
        assert np.linalg.norm(c[~geo.disc_b[led]]) < 1e-3 * np.linalg.norm(c)   # aliasing floor only
        s4 = O.kk_field(truth.clean[led], p.kappa_bright[led], pad=4)
        c4 = np.fft.fftshift(O.sub_spectrum(s4))
        assert np.linalg.norm(c4[~geo.disc_b[led]]) < 1e-12 * np.linalg.norm(c4)
        assert abs(c4[32, 32].imag) < 1e-13 * abs(c4[32, 32])


def test_fourier_resample_preserves_samples_and_inverts():
    rng = np.random.default_rng(0)
    cfg = get_config(0)
    _, truth = make_tile(cfg, 0, keep_clean=True)
    a = truth.clean[0]
    up = O.fourier_resample(a, 128)
    assert np.abs(up[::2, ::2] - a).max() < 1e-12
    assert np.abs(up.imag).max() < 1e-12
    assert np.abs(O.fourier_resample(up, 64) - a).max() < 1e-12
