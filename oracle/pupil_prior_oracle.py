"""fp64 CPU oracle of the slide-level pupil prior.

TEST INFRASTRUCTURE - not part of the product path; shares no code with the CUDA library.

The paper shows the recovered pupil varying smoothly from region to region of a slide (Fig. 4(b)) and
states no algorithm that uses it.  Reading B9: the Zernike coefficients recovered per tile are
fitted, coefficient by coefficient, by a polynomial of total degree <= `order` in the tile's slide coordinates
(X, Y), by unweighted least squares over the tiles whose reconstruction succeeded (status 0).  The fit evaluated at a
tile is that tile's PRIOR: it replaces the gradient-domain start of the aberration fit
(`apic_oracle.solve_aberration(..., c_init=...)`), which rescues tiles whose own start lands in a wrong minimum of
the re-wrapped fit (R11) and leaves every other tile's result unchanged.

Terms, in this order: 1, X, Y, X^2, XY, Y^2 (the first 1 / 3 / 6 for order 0 / 1 / 2).  If the tiles that succeeded
do not determine the polynomial (numerical rank of the design matrix below the number of terms) the fit falls back
to order 0 (the mean over those tiles), and to all zeros if no tile succeeded.

Pins (tests/test_oracle_pupil_prior.py): the seeded generator's quadratic field (apic_synth, an independent formula)
is recovered to 1e-12 including at tiles that were excluded; garbage at failed tiles is ignored; order 0 is the mean;
the fallbacks; averaging reduces independent per-tile noise by ~sqrt(terms / tiles).
"""
from __future__ import annotations

import numpy as np

N_TERMS = {0: 1, 1: 3, 2: 6}


def design_matrix(xy: np.ndarray, order: int) -> np.ndarray:
    """[tiles][n_terms]: 1, X, Y, X^2, XY, Y^2 truncated to the order."""
    x, y = np.asarray(xy, dtype=np.float64).T
    cols = [np.ones_like(x), x, y, x * x, x * y, y * y]
    return np.stack(cols[:N_TERMS[order]], axis=1)


def pupil_field_fit(coefs: np.ndarray, status: np.ndarray, xy: np.ndarray, order: int = 2):
    """coefs [tiles][n_z], status [tiles] (0 = use), xy [tiles][2].  Returns (fit [tiles][n_z], poly [6][n_z]; unused
    terms are 0)."""
    coefs = np.asarray(coefs, dtype=np.float64)
    ok = np.asarray(status) == 0
    nz = coefs.shape[1]
    poly = np.zeros((6, nz))
    if ok.any():
        b = design_matrix(xy, order)
        if np.linalg.matrix_rank(b[ok]) == b.shape[1]:
            sol, *_ = np.linalg.lstsq(b[ok], coefs[ok], rcond=None)
            poly[:b.shape[1]] = sol
        else:
            poly[0] = coefs[ok].mean(axis=0)
    return design_matrix(xy, 2) @ poly, poly
