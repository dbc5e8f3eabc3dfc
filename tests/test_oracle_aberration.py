"""Pins for the aberration extraction O4 (Eq. 8-10) and stitching O5 (:116)."""
import dataclasses
import math

import numpy as np
import pytest

from apic_synth import get_config, make_tile
from apic_synth.forward import object_spectrum_raw, pupil_phase_at
from oracle import apic_oracle as O
from helpers import oracle_params, read_golden_table, rel_l2, truth_object_spectrum


def _golden(key):
    for row in read_golden_table("geometry_counts.txt"):
        if row[0] == key:
            return row
    raise KeyError(key)


def _true_spectra(cfg, truth, geo):
    """S_hat_i e^{-j theta_i} := O(k) H(k+kappa_i) e^{-j phi(kappa_i)} on D_i, centred (Eq. 7)."""
    out = []
    o = object_spectrum_raw(cfg, truth.obj)
    for kap in geo.kappa_b:
        mask, phi = pupil_phase_at(cfg, truth.coef, kap)
        _, phi0 = pupil_phase_at(cfg, truth.coef, kap)          # phi(k+kappa) incl. k = 0
        theta = phi0[0, 0] + np.angle(o[0, 0])                   # KK also removes arg O(0)
        out.append(np.fft.fftshift(np.where(mask, o * np.exp(1j * (phi - theta)), 0.0)))
    return out


@pytest.mark.parametrize("key,idx", [("cfg0", 0), ("cfg1_2_4", 2), ("cfg3", 3)])
def test_row_counts_match_survey(key, idx):
    g = _golden(key)
    cfg = get_config(idx)
    geo = O.Geometry(oracle_params(cfg))
    assert len(geo.pairs) == int(g[4])
    rows = grows = 0
    for i, l in geo.pairs:
        m = geo.disc_b[i] & geo.disc_b[l]
        rows += int(m.sum())
        grows += int((m[:, :-1] & m[:, 1:]).sum() + (m[:-1, :] & m[1:, :]).sum())
    assert rows == int(g[5]) and grows == int(g[6])
    union = np.zeros_like(geo.disc_b[0])
    for m in geo.disc_b:
        union |= m
    assert int(union.sum()) == int(g[7])
    if g[8] != "-":
        for m in geo.disc_d:
            union |= m
        assert int(union.sum()) == int(g[8])


def test_opposite_discs_touch_only_at_dc_and_are_dropped():
    geo = O.Geometry(oracle_params(get_config(0)))
    assert (0, 2) not in geo.pairs and (1, 3) not in geo.pairs
    assert int((geo.disc_b[0] & geo.disc_b[2]).sum()) == 1


def test_defocus_column_closed_form_and_null_columns():
    cfg = get_config(1)
    p = oracle_params(cfg)
    p.noll = [1, 2, 3, 4]
    geo = O.Geometry(p)
    for (i, l) in geo.pairs[:6]:
        mask, iy, ix, a = O.aberration_rows(geo, i, l)
        kx, ky = geo.kx[iy, ix], geo.ky[iy, ix]
        dk = geo.kappa_b[i] - geo.kappa_b[l]
        closed = 4 * math.sqrt(3) * (kx * dk[0] + ky * dk[1]) / geo.radius ** 2
        assert np.abs(a[:, 3] - closed).max() < 1e-11          # beta for defocus is linear in K
        assert np.abs(a[:, :3]).max() < 1e-12                  # piston and both tilts cancel (R9)


@pytest.mark.parametrize("idx,scale", [(0, 1.0), (0, 3.0), (1, 1.0), (1, 2.0)])
def test_exact_coefficients_from_true_spectra_despite_wrapping(idx, scale):
    cfg = get_config(idx)
    cfg = dataclasses.replace(cfg, pupil_strength=cfg.pupil_strength * scale)
    _, truth = make_tile(cfg, 0, noise="none")
    p = oracle_params(cfg)
    geo = O.Geometry(p)
    spectra = _true_spectra(cfg, truth, geo)
    c, status, info = O.solve_aberration(geo, spectra, refine_iters=3)
    ct = np.array([truth.coef[j] for j in cfg.noll_fit])
    assert status == O.STATUS_OK
    assert np.abs(c - ct).max() < 1e-11
    assert info["residual_rms"] < 1e-11
    # the wrapped one-shot linear solve of the paper is NOT enough here (R11): |beta| exceeds pi
    a = np.concatenate([O.aberration_rows(geo, i, l)[3] for i, l in geo.pairs])
    assert np.abs(a @ ct).max() > math.pi


def test_stitch_equals_truth_on_union_with_true_inputs():
    cfg = get_config(1)
    _, truth = make_tile(cfg, 0, noise="none")
    p = oracle_params(cfg)
    geo = O.Geometry(p)
    spectra = _true_spectra(cfg, truth, geo)
    ct = np.array([truth.coef[j] for j in cfg.noll_fit])
    o_hat, known = O.stitch(geo, spectra, ct)
    target = truth_object_spectrum(cfg, truth, geo.radius)
    assert rel_l2(o_hat[known], target[known]) < 1e-12
    assert np.all(o_hat[~known] == 0)
    assert abs(o_hat[cfg.tile_n // 2, cfg.tile_n // 2].imag) < 1e-14


def test_end_to_end_brightfield_noise_free():
    """KK -> aberration -> stitch on clean fp64 data, pad 2: coefficients <= 1e-6 rad (contract:
    < 1e-3), spectrum equals truth on the union of discs up to R9/R14."""
    cfg = get_config(0)
    _, truth = make_tile(cfg, 0, keep_clean=True)
    p = oracle_params(cfg, kk_pad=2)
    r = O.reconstruct_tile(truth.clean, p, keep=True)
    ct = np.array([truth.coef[j] for j in cfg.noll_fit])
    assert r.status == O.STATUS_OK
    assert np.linalg.norm(r.zernike - ct) < 1e-6
    target = truth_object_spectrum(cfg, truth, p.radius)
    assert rel_l2(r.o_hat[r.known], target[r.known]) < 1e-6
    # field on the 2x grid equals the band-limited ground truth (same check in real space)
    assert rel_l2(r.field, O.output_field(np.where(r.known, target, 0), 2)) < 1e-6


def test_config1_with_read_noise_meets_contract():
    cfg = get_config(1)
    stack, truth = make_tile(cfg, 0)
    r = O.reconstruct_tile(stack, oracle_params(cfg), keep=True)
    ct = np.array([truth.coef[j] for j in cfg.noll_fit])
    assert r.status == O.STATUS_OK
    assert np.linalg.norm(r.zernike - ct) < 1e-3              # BASELINE.json: < 1e-3 rad RMS
    assert r.info["rows"] == 33096 and r.info["grad_rows"] == 64144


def test_solver_flags_hopeless_phase_data():
    cfg = get_config(0)
    geo = O.Geometry(oracle_params(cfg))
    rng = np.random.default_rng(5)
    junk = [rng.standard_normal((64, 64)) + 1j * rng.standard_normal((64, 64)) for _ in range(4)]
    _, status, info = O.solve_aberration(geo, junk, refine_iters=3)
    assert status == O.STATUS_SOLVE_FAILED and info["residual_rms"] > 1.0
