"""CPU-side checks of the boundary (no compute calls): libapic.so loads, exports every symbol that
include/apic.h declares, its host-only fp64 geometry reproduces the index-set sizes that geometry
alone fixes (tests/golden/geometry_counts.txt, numbers printed in SURVEY.md §8, produced by an
implementation independent of both the oracle and the library), parameter validation returns
APIC_EINVAL, and the product path fails loudly (APIC_ECUDA) when no CUDA device exists."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from apic_synth import get_config, led_kvectors
from helpers import plan_from_config, read_golden_table

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def A():
    import paper_2407_20469_b200 as pkg
    if not pkg.LIB_PATH.exists():
        from paper_2407_20469_b200.build import build
        build()
    pkg.load()
    return pkg


def _params(A, cfg, **opts):
    kb, kd = led_kvectors(cfg)
    return A.make_params(cfg.tile_n, cfg.upsample, cfg.wavelength_um, cfg.pixel_um, cfg.na_obj, kb, kd,
                         cfg.noll_fit, **opts)


def test_every_declared_symbol_is_exported(A):
    text = open(os.path.join(ROOT, "include", "apic.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(apic_[a-z0-9_]+)\s*\(", text))
    assert {"apic_plan_create", "apic_reconstruct", "apic_plan_destroy"} <= declared
    lib = A.load()
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in apic.h but not exported by libapic.so"
    assert set(A.EXPORTS) == declared


def test_struct_layout_matches_header(A):
    """apic_params_default must fill the ctypes mirror consistently (catches field-order drift)."""
    p = A.ApicParams()
    A.load().apic_params_default(C.byref(p))
    assert (p.kk_pad, p.refine_iters, p.df_iters, p.max_batch, p.bg_mode, p.chunk_tiles) == (1, 3, 48, 64, 0, 0)
    assert p.intensity_floor == pytest.approx(1e-6) and p.df_tol == pytest.approx(1e-4)


@pytest.mark.parametrize("key,index", [("cfg0", 0), ("cfg1_2_4", 2), ("cfg3", 3)])
def test_host_geometry_counts_match_golden(A, key, index):
    rows = {r[0]: r for r in read_golden_table("geometry_counts.txt")}
    g = rows[key]
    cfg = get_config(index)
    p, keep = _params(A, cfg)
    info, dark = A.geometry_info(p)
    assert info["n_pairs"] == int(g[4])
    assert info["n_rows"] == int(g[5])
    assert info["n_grad_rows"] == int(g[6])
    assert info["n_union"] == int(g[7])
    if g[8] != "-":
        assert info["n_known"] == int(g[8])
    if g[9] != "-":
        assert dark[0] == (0, int(g[9]), int(g[10]))
        ring2 = [d for d in dark if d[0] == 8][0]
        assert ring2[1:] == (int(g[11]), int(g[12]))
    assert info["radius_bins"] == pytest.approx(0.25 * cfg.tile_n * 0.345 / 0.52, rel=1e-12)


def test_darkfield_order_is_ascending_illumination_na(A):
    cfg = get_config(2)
    p, keep = _params(A, cfg)
    _, dark = A.geometry_info(p)
    assert [d[0] for d in dark] == list(range(16))            # ring 0.30 (LEDs 0-7) before ring 0.40
    cfg3 = get_config(3, tile_n=128)
    p3, keep3 = _params(A, cfg3)
    info3, dark3 = A.geometry_info(p3)
    assert info3["n_dark_used"] == 32 and [d[0] for d in dark3] == list(range(32))


def test_invalid_parameters_are_rejected(A):
    lib = A.load()
    info = A.PlanInfo()
    cfg = get_config(0)

    def rc(tile_n=cfg.tile_n, upsample=cfg.upsample, noll=cfg.noll_fit, kb=None, kd=None):
        kb0, kd0 = led_kvectors(cfg)
        p, keep = A.make_params(tile_n, upsample, cfg.wavelength_um, cfg.pixel_um, cfg.na_obj,
                                kb0 if kb is None else kb, kd0 if kd is None else kd, noll)
        return lib.apic_geometry_info(C.byref(p), C.byref(info), None, None, None, 0)

    kb, _ = led_kvectors(cfg)
    assert rc() == A.APIC_OK
    assert rc(tile_n=96) == A.APIC_EINVAL                      # not a supported power of two
    assert rc(upsample=5) == A.APIC_EINVAL
    assert rc(noll=[3, 4, 5]) == A.APIC_EINVAL                 # tilt is in the null space of Eq. 10 (R9)
    assert rc(noll=[4, 4]) == A.APIC_EINVAL
    assert rc(kb=kb * 1.2) == A.APIC_EINVAL                    # NA-matching condition violated
    assert rc(kd=kb * 0.5) == A.APIC_EINVAL                    # "darkfield" LED inside the pupil
    assert rc(kd=kb * 2.2) == A.APIC_EINVAL                    # synthetic aperture leaves the raw grid
    assert b"" != lib.apic_strerror(A.APIC_EINVAL)


def test_unknown_fraction_bound_of_the_paper(A):
    """at most 42 % of a darkfield LED's disc may be unknown."""
    cfg = get_config(0)
    kb, _ = led_kvectors(cfg)
    lib = A.load()
    info = A.PlanInfo()
    ok, keep = A.make_params(64, 2, cfg.wavelength_um, cfg.pixel_um, cfg.na_obj, kb, kb[:1] * 1.2, cfg.noll_fit)
    assert lib.apic_geometry_info(C.byref(ok), C.byref(info), None, None, None, 0) == A.APIC_OK
    far, keep2 = A.make_params(64, 2, cfg.wavelength_um, cfg.pixel_um, cfg.na_obj, kb, kb[:1] * 1.9, cfg.noll_fit)
    assert lib.apic_geometry_info(C.byref(far), C.byref(info), None, None, None, 0) == A.APIC_EINVAL
    assert b"unknown fraction" in lib.apic_strerror(A.APIC_EINVAL)


def test_no_cpu_fallback(A):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    cfg = get_config(0)
    with pytest.raises(A.ApicError, match="CUDA"):
        plan_from_config(A, cfg)


def test_ring_wise_order_index_sets_match_the_oracle(A):
    """df_order 1 (reading R15b): the library's |U|, |Q| per LED equal those of the oracle's dark_order='ring'
    (independent code: run-length Minkowski differences here, all-pairs differences there), and its reduced grids
    are alias-free for those sets."""
    from oracle import apic_oracle as O
    from helpers import oracle_params
    for cfg in (get_config(2), get_config(2, tile_n=64, batch=1, grid=(1, 1))):
        p, keep = _params(A, cfg, df_order=1)
        _, dark = A.geometry_info(p)
        sets, _ = O.darkfield_sets(O.Geometry(oracle_params(cfg, dark_order="ring")))
        assert [(d.led, int(d.U.sum()), int(d.Q.sum())) for d in sets] == dark
        seq = A.geometry_info(_params(A, cfg)[0])[1]
        assert dark[0] == seq[0] and dark[8] == seq[8] and sum(d[1] for d in dark) > sum(d[1] for d in seq)
        n = cfg.tile_n
        for (mx, my), ds in zip(A.geometry_dark_grids(p), sets):
            for m, axis in ((mx, 1), (my, 0)):
                u, pp, q = (np.nonzero(mm.any(axis=1 - axis))[0] for mm in (ds.U, ds.P, ds.Q))
                ext = max(abs(int(u.max() - pp.min() - (q.min() - n // 2))), abs(int(u.min() - pp.max() - (q.max() - n // 2))))
                assert m > ext


@pytest.mark.parametrize("index,tile_n", [(2, 256), (3, 256), (2, 64)])
def test_reduced_darkfield_grids_are_alias_free(A, index, tile_n):
    """The library's per-LED cyclic grid (mx, my) for the CG mat-vecs of Eq. 13 must exceed, per axis,
    the extent of the lag set U - P - Q computed from the ORACLE's index sets (then no wrong pair
    u - p = k + (a mx, b my) exists), and must hold the disc and Q without folding."""
    from oracle import apic_oracle as O
    from helpers import oracle_params
    cfg = get_config(index, tile_n=tile_n, batch=1, grid=(1, 1)) if tile_n != get_config(index).tile_n else get_config(index)
    p, keep = _params(A, cfg)
    grids = A.geometry_dark_grids(p)
    geo = O.Geometry(oracle_params(cfg))
    sets, _ = O.darkfield_sets(geo)
    assert len(grids) == len(sets)
    allowed = {3 * tile_n // 8, tile_n // 2, 5 * tile_n // 8, 3 * tile_n // 4, tile_n}
    smaller = 0
    for (mx, my), ds in zip(grids, sets):
        assert mx in allowed and my in allowed
        ext = []
        for axis in (1, 0):
            u, pp, q = (np.nonzero(m.any(axis=1 - axis))[0] for m in (ds.U, ds.P, ds.Q))
            hi = u.max() - pp.min() - (q.min() - tile_n // 2)
            lo = u.min() - pp.max() - (q.max() - tile_n // 2)
            ext.append(max(abs(int(hi)), abs(int(lo))))
        assert mx > ext[0] and my > ext[1], (ds.led, mx, my, ext)
        smaller += mx * my < tile_n * tile_n
    if index == 2:
        assert smaller == len(sets)            # config 2: every LED runs on a reduced grid
