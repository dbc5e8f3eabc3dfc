"""Helpers shared by the oracle pins and the GPU parity tests (no method arithmetic)."""
import os

import numpy as np

from apic_synth import led_kvectors
from apic_synth.forward import object_spectrum_raw, truth_zernike
from oracle import apic_oracle as O

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def oracle_params(cfg, **kw) -> O.OracleParams:
    kb, kd = led_kvectors(cfg)
    return O.OracleParams(tile_n=cfg.tile_n, upsample=cfg.upsample, wavelength_um=cfg.wavelength_um,
                          pixel_um=cfg.pixel_um, na_obj=cfg.na_obj, k_bright=kb, k_dark=kd,
                          noll=list(cfg.noll_fit), **kw)


def plan_from_config(A, cfg, **opts):
    """apic_plan for an apic_synth config (optics, LED layout and fitted Noll terms of the recipe)."""
    from apic_synth import plan_args
    return A.Plan(*plan_args(cfg), **opts)


def truth_object_spectrum(cfg, truth, radius):
    """What the reconstruction must equal inside the synthetic band:
    O_true(k) * exp(j*tilt(k)) * exp(-j*arg O_true(0)), centred [N][N]; a pupil tilt (Noll 2, 3)
    is exactly a sub-pixel object shift and piston is the global phase."""
    n = cfg.tile_n
    o = np.fft.fftshift(object_spectrum_raw(cfg, truth.obj))
    c = np.arange(n) - n // 2
    kx, ky = np.meshgrid(c, c, indexing="xy")
    tilt = np.zeros((n, n))
    for j in (2, 3):
        if truth.coef.get(j, 0.0) != 0.0:
            tilt += truth.coef[j] * truth_zernike(j, kx / radius, ky / radius)
    return o * np.exp(1j * tilt) * np.exp(-1j * np.angle(o[n // 2, n // 2]))


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b)))


def read_golden_table(name):
    """Whitespace table with '#' comments -> list of rows of strings."""
    rows = []
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows
