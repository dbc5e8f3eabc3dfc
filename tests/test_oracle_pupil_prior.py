"""Pins of the slide-level pupil prior (reading B9): oracle/pupil_prior_oracle.py and
the c_init argument of apic_oracle.solve_aberration.  Expected values come from the generator's own field polynomial
(an independent formula), from closed forms and from the truth of noise-free forward data."""
import numpy as np

from apic_synth import get_config, make_tile
from apic_synth.forward import truth_coefficients
from oracle import apic_oracle as O
from oracle import pupil_prior_oracle as P
from helpers import oracle_params
from test_oracle_aberration import _true_spectra


def _grid_xy(gx, gy):
    xs = -1.0 + (2.0 * np.arange(gx) + 1.0) / gx
    ys = -1.0 + (2.0 * np.arange(gy) + 1.0) / gy
    X, Y = np.meshgrid(xs, ys, indexing="xy")
    return np.stack([X.ravel(), Y.ravel()], axis=1)


def test_generators_quadratic_pupil_field_is_recovered_exactly():
    cfg = get_config(2)                                       # 8 x 8 tiles, coefficients quadratic in the tile's (X, Y)
    truth = np.array([[truth_coefficients(cfg, t, np.random.default_rng(0))[j] for j in cfg.noll_truth] for t in range(cfg.batch)])
    xy = _grid_xy(*cfg.grid)
    status = np.zeros(cfg.batch, dtype=np.int32)
    rng = np.random.default_rng(0)
    bad = rng.choice(cfg.batch, 20, replace=False)
    status[bad] = rng.choice([1, 2, 3], 20)
    coefs = truth.copy()
    coefs[bad] = 1e3 * rng.standard_normal((20, truth.shape[1]))     # garbage where the reconstruction did not succeed
    fit, poly = P.pupil_field_fit(coefs, status, xy, 2)
    assert np.abs(fit - truth).max() < 1e-12                  # also at the 20 excluded tiles
    assert np.abs(fit[bad] - truth[bad]).max() < 1e-12
    # a linear fit cannot represent it: the test above is not vacuous
    fit1, _ = P.pupil_field_fit(coefs, status, xy, 1)
    assert np.abs(fit1 - truth).max() > 1e-3


def test_order_zero_is_the_mean_and_the_fallbacks():
    rng = np.random.default_rng(1)
    c = rng.standard_normal((10, 4))
    xy = rng.uniform(-1, 1, (10, 2))
    st = np.array([0, 0, 3, 0, 1, 0, 0, 2, 0, 0])
    fit, poly = P.pupil_field_fit(c, st, xy, 0)
    assert np.allclose(fit, c[st == 0].mean(axis=0)[None, :], atol=1e-15) and not poly[1:].any()
    # three tiles cannot determine six terms: mean of those three
    st3 = np.array([0, 3, 3, 0, 3, 3, 3, 3, 0, 3])
    fit, poly = P.pupil_field_fit(c, st3, xy, 2)
    assert np.allclose(fit, c[st3 == 0].mean(axis=0)[None, :], atol=1e-15)
    # collinear tiles (one scan row) cannot determine the Y terms either
    xy_row = np.stack([np.linspace(-1, 1, 10), np.zeros(10)], axis=1)
    fit, poly = P.pupil_field_fit(c, np.zeros(10, int), xy_row, 2)
    assert np.allclose(fit, c.mean(axis=0)[None, :], atol=1e-15)
    fit, poly = P.pupil_field_fit(c, np.full(10, 3), xy, 2)
    assert not fit.any() and not poly.any()


def test_fit_averages_independent_noise():
    xy = _grid_xy(16, 16)
    q = np.array([0.3, -0.2, 0.1, 0.05, -0.07, 0.02])
    clean = (P.design_matrix(xy, 2) @ q)[:, None]
    rng = np.random.default_rng(2)
    noisy = clean + 1e-2 * rng.standard_normal(clean.shape)
    fit, poly = P.pupil_field_fit(noisy, np.zeros(256, int), xy, 2)
    rms = np.sqrt(np.mean((fit - clean) ** 2))
    assert rms < 1e-2 * np.sqrt(6 / 256) * 1.5 and np.abs(poly[:, 0] - q).max() < 1e-2


def test_prior_replaces_the_gradient_start_and_rescues_a_wrong_minimum():
    """Config-3 strength on a 128-pixel tile is outside the basin of the gradient-domain start (R11): from exact
    spectra the default fit lands 0.4 rad from the truth.  Started from a prior within 50 % of the truth the same
    refinement reaches the truth; where the default start works (N = 256) the prior changes nothing."""
    cfg = get_config(3, tile_n=128, batch=1, grid=(1, 1))
    _, truth = make_tile(cfg, 0, noise="none")
    geo = O.Geometry(oracle_params(cfg))
    spectra = _true_spectra(cfg, truth, geo)
    ct = np.array([truth.coef[j] for j in cfg.noll_fit])
    c0, st0, _ = O.solve_aberration(geo, spectra, 3)
    assert np.abs(c0 - ct).max() > 0.1
    for f in (1.0, 0.8, 0.5):
        c, st, info = O.solve_aberration(geo, spectra, 3, c_init=f * ct)
        assert st == O.STATUS_OK and np.abs(c - ct).max() < 1e-11 and info["residual_rms"] < 1e-11
    cfg = get_config(1)
    _, truth = make_tile(cfg, 0, noise="none")
    geo = O.Geometry(oracle_params(cfg))
    spectra = _true_spectra(cfg, truth, geo)
    ct = np.array([truth.coef[j] for j in cfg.noll_fit])
    c_def, _, _ = O.solve_aberration(geo, spectra, 3)
    c_pri, _, _ = O.solve_aberration(geo, spectra, 3, c_init=0.7 * ct)
    assert np.abs(c_def - ct).max() < 1e-11 and np.abs(c_pri - ct).max() < 1e-11
    # a hopeless prior is flagged by the unchanged status rule
    rng = np.random.default_rng(3)
    _, st_bad, info = O.solve_aberration(geo, spectra, 3, c_init=ct + 3.0 * rng.standard_normal(ct.size))
    assert st_bad == O.STATUS_SOLVE_FAILED or np.isfinite(info["residual_rms"])
