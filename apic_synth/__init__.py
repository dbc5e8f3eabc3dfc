"""Seeded synthetic inputs for the APIC reconstruction path.

This package is the ONLY code shared by the fp64 CPU oracle's tests and the CUDA
path's tests/bench: it makes intensity stacks with the paper's forward model
(Eq. 1-2, in the DC-centred frame of Eq. 3) and
holds none of the reconstruction arithmetic.  It imports neither ``oracle`` nor
``paper_2407_20469_b200``.
"""
from .configs import ApicConfig, get_config, led_kvectors, plan_args, CONFIG_NAMES  # noqa: F401
from .forward import make_tile, make_batch, TileTruth  # noqa: F401
