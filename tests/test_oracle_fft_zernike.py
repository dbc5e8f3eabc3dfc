"""Pins for the oracle's transforms and Zernike basis (SURVEY.md §8(c) "FFT", R9)."""
import math

import numpy as np
import pytest

from apic_synth.forward import noll_table, truth_zernike
from oracle import apic_oracle as O
from helpers import read_golden_table


def test_naive_dft_matches_fft_at_64():
    rng = np.random.default_rng(1)
    a = rng.standard_normal((64, 64)) + 1j * rng.standard_normal((64, 64))
    ref = O.naive_dft2(a)                      # the definition
    assert np.abs(O.fft2n(a) * 64 * 64 - ref).max() < 1e-10
    assert np.abs(O.ifft2u(a) - O.naive_dft2(a, inverse=True)).max() < 1e-10


def test_fft_single_bin_closed_form():
    # one spatial harmonic e^{+j 2 pi (3x - 5y)/N} has exactly one coefficient, = 1, at (kx,ky)=(3,-5)
    n = 64
    x = np.arange(n)
    s = np.exp(1j * 2 * np.pi * (3 * x[None, :] - 5 * x[:, None]) / n)
    spec = O.fft2n(s)
    k = O.signed_bins(n)
    iy, ix = int(np.nonzero(k == -5)[0][0]), int(np.nonzero(k == 3)[0][0])
    assert abs(spec[iy, ix] - 1.0) < 1e-13
    spec[iy, ix] = 0
    assert np.abs(spec).max() < 1e-13


def test_parseval_and_round_trip():
    rng = np.random.default_rng(2)
    a = rng.standard_normal((128, 128)) + 1j * rng.standard_normal((128, 128))
    spec = O.fft2n(a)
    assert abs((np.abs(a) ** 2).mean() - (np.abs(spec) ** 2).sum()) < 1e-10
    assert np.abs(O.ifft2u(spec) - a).max() < 1e-12


def test_noll_table_matches_literature():
    for j, n, m in read_golden_table("noll_table.txt"):
        assert O.noll_to_nm(int(j)) == (int(n), int(m))


def test_noll_closed_form_matches_enumeration_to_66():
    tab = noll_table(66)
    for j in range(1, 67):
        assert O.noll_to_nm(j) == tab[j]


def test_zernike_closed_forms():
    rho = np.linspace(0, 1.05, 23)
    th = np.linspace(-3, 3, 23)
    assert np.allclose(O.zernike(4, rho, th), math.sqrt(3) * (2 * rho ** 2 - 1))
    assert np.allclose(O.zernike(5, rho, th), math.sqrt(6) * rho ** 2 * np.sin(2 * th))
    assert np.allclose(O.zernike(6, rho, th), math.sqrt(6) * rho ** 2 * np.cos(2 * th))
    assert np.allclose(O.zernike(7, rho, th), math.sqrt(8) * (3 * rho ** 3 - 2 * rho) * np.sin(th))
    assert np.allclose(O.zernike(8, rho, th), math.sqrt(8) * (3 * rho ** 3 - 2 * rho) * np.cos(th))
    assert np.allclose(O.zernike(11, rho, th), math.sqrt(5) * (6 * rho ** 4 - 6 * rho ** 2 + 1))
    assert np.allclose(O.zernike(2, rho, th), 2 * rho * np.cos(th))
    assert np.allclose(O.zernike(3, rho, th), 2 * rho * np.sin(th))


def test_zernike_orthonormal_on_unit_disc():
    # Gauss-Legendre in rho^2 x uniform in theta integrates polynomials of this degree exactly
    nr, nt = 40, 128
    x, w = np.polynomial.legendre.leggauss(nr)
    t = 0.5 * (x + 1)                       # t = rho^2 in [0,1], weight w/2
    rho = np.sqrt(t)
    th = 2 * np.pi * np.arange(nt) / nt
    R, T = np.meshgrid(rho, th, indexing="ij")
    W = np.repeat((w / 2)[:, None], nt, axis=1) / nt     # integral over disc / pi
    js = list(range(1, 38))
    Z = np.stack([O.zernike(j, R, T) for j in js])
    gram = np.einsum("irt,jrt,rt->ij", Z, Z, W)
    assert np.abs(gram - np.eye(len(js))).max() < 1e-10


def test_oracle_zernike_equals_generator_zernike():
    # two different formulas (factorial sum vs Jacobi polynomials) for the same basis
    rng = np.random.default_rng(3)
    x = rng.uniform(-1, 1, 500)
    y = rng.uniform(-1, 1, 500)
    for j in range(1, 38):
        a = O.zernike(j, np.hypot(x, y), np.arctan2(y, x))
        assert np.abs(a - truth_zernike(j, x, y)).max() < 1e-9
