"""Writes tests/golden/cfg3_tile0.npz: the oracle's result for tile 0 of BASELINE.json config 3 at its
stated size (N = 512, 12 NA-matching + 32 darkfield LEDs to NA_ill 0.45, 34 fitted Zernike terms, 1 rad
RMS pupil, Poisson noise; PAPER.md:171 512^2 patches, :153 LED layout).

Calls ONLY `oracle/` and the seeded generator `apic_synth/` (never the CUDA library).  The dense
`lstsq` of Eq. 13 at N = 512 (up to 37,000 x 4,786 complex128 per LED) takes minutes per tile on a few
cores, which is why the result is stored instead of recomputed by the GPU parity test.

    python tests/golden/make_cfg3_golden.py            # tile 0: about 7 min on 4 cores, <= 20 GB of memory
    python tests/golden/make_cfg3_golden.py 1 2 3 4 5 6 7    # more tiles (>= 8 tiles of config 3)

cfg3_tile0.npz holds everything; cfg3_tile<t>.npz for t > 0 hold only what differs from tile to tile (spectrum on the
known region, coefficients, status, field sample): the index arrays are geometry and are read from tile 0's file.

Stored (complex64 / float64): the object spectrum on the final known region (row-major order of the
centred mask), the Zernike coefficients, the status, |U| and |Q| per darkfield LED in processing order,
the index of every known bin and which step solved it (-1: NA-matching union, k: k-th darkfield LED), so
that the test needs no oracle geometry at N = 512 and can compare band by band.
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
sys.path.insert(0, os.path.dirname(HERE))

from apic_synth import get_config, make_tile      # noqa: E402
from oracle import apic_oracle as O               # noqa: E402
from helpers import oracle_params                 # noqa: E402


def main(tiles):
    cfg = get_config(3)
    t0 = time.time()
    p = oracle_params(cfg)
    geo = O.Geometry(p)
    sets, known_final = O.darkfield_sets(geo)
    print(f"geometry {time.time() - t0:.0f} s: {len(sets)} darkfield LEDs, |known| = {int(known_final.sum())}", flush=True)
    for tile in tiles:
        stack, _ = make_tile(cfg, tile)
        r = O.reconstruct_tile(stack, p, geo=geo, sets=sets, keep=True)
        print(f"tile {tile}: oracle {time.time() - t0:.0f} s, status {r.status}", flush=True)
        if tile == 0:
            write_full(geo, sets, r)
        else:
            assert np.array_equal(r.known, known_final)
            np.savez_compressed(os.path.join(HERE, f"cfg3_tile{tile}.npz"),
                                o_hat_known=r.o_hat[r.known].astype(np.complex64),
                                zernike=np.asarray(r.zernike, dtype=np.float64), status=np.int32(r.status),
                                field_sample=r.field[::64, ::64].astype(np.complex64))
        print(f"tile {tile} written", flush=True)


def write_full(geo, sets, r):
    ky, kx = np.nonzero(r.known)
    owner = np.full(r.known.shape, -1, dtype=np.int8)       # -1: union of the NA-matching discs; k: solved by the k-th darkfield LED
    for k, ds in enumerate(sets):
        owner[ds.U] = k
    np.savez_compressed(
        os.path.join(HERE, "cfg3_tile0.npz"),
        o_hat_known=r.o_hat[r.known].astype(np.complex64),
        known_iy=ky.astype(np.int16), known_ix=kx.astype(np.int16),
        owner=owner[r.known],
        kappa_dark=np.asarray(geo.kappa_d, dtype=np.float64),
        zernike=np.asarray(r.zernike, dtype=np.float64),
        status=np.int32(r.status),
        led=np.array([s.led for s in sets], dtype=np.int32),
        n_unknown=np.array([int(s.U.sum()) for s in sets], dtype=np.int32),
        n_equations=np.array([int(s.Q.sum()) for s in sets], dtype=np.int32),
        field_sample=r.field[::64, ::64].astype(np.complex64),
    )


if __name__ == "__main__":
    main([int(a) for a in sys.argv[1:]] or [0])
