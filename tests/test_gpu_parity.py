"""GPU parity: libapic (through the C ABI) against the fp64 oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json's: relative L2 <= 1e-4 on the complex field and
<= 1e-3 rad RMS on the recovered pupil phase (= ||c_gpu - c_oracle||_2 over the fitted Noll terms,
which have unit RMS on the disc; R9).  The output's global phase is fixed by construction
(DC real-positive, R14), so no alignment is applied.  Integer outputs (status) must be equal."""
import numpy as np
import pytest

from apic_synth import get_config, make_batch
from oracle import apic_oracle as O
from helpers import oracle_params, rel_l2

pytestmark = pytest.mark.gpu

FIELD_TOL = 1e-4      # BASELINE.json north_star
PUPIL_TOL = 1e-3      # rad RMS


@pytest.fixture(scope="module")
def A():
    import torch
    assert torch.cuda.is_available()
    import paper_2407_20469_b200 as pkg
    pkg.load()                                   # raises if libapic.so is missing: no fallback
    return pkg


def gpu_reconstruct(A, cfg, stacks, **opts):
    import torch
    opts.setdefault("max_batch", len(stacks))
    plan = A.Plan.from_config(cfg, **opts)
    x = torch.from_numpy(np.ascontiguousarray(stacks)).cuda()
    field, zern, pupil, status = plan.reconstruct(x)
    torch.cuda.synchronize()
    return plan, field.cpu().numpy(), zern.cpu().numpy(), pupil.cpu().numpy(), status.cpu().numpy()


def oracle_reconstruct(cfg, stacks, **kw):
    p = oracle_params(cfg, **kw)
    geo = O.Geometry(p)
    sets = O.darkfield_sets(geo)[0] if cfg.n_dark else None
    return [O.reconstruct_tile(s, p, geo=geo, sets=sets, keep=True) for s in stacks], geo


def check_tile(ref, field, zern, pupil, status, label):
    assert int(status) == ref.status, f"{label}: status {status} != oracle {ref.status}"
    e_f = rel_l2(field, ref.field)
    e_c = float(np.linalg.norm(zern - ref.zernike))
    mask = np.abs(ref.pupil) > 0
    e_p = float(np.sqrt(np.mean(np.angle(pupil[mask] * np.conj(ref.pupil[mask])) ** 2)))
    assert e_f <= FIELD_TOL, f"{label}: field rel L2 {e_f:.3e}"
    assert e_c <= PUPIL_TOL and e_p <= PUPIL_TOL, f"{label}: pupil {e_c:.3e} / {e_p:.3e} rad"
    assert np.array_equal(np.abs(pupil) > 0.5, mask), f"{label}: pupil support"
    return e_f, e_c


# ---------------------------------------------------------------------------------- kernel K1
@pytest.mark.parametrize("n", [64, 128, 256, 512])
def test_fft2d_matches_oracle_transform(A, n):
    import torch
    rng = np.random.default_rng(n)
    x = (rng.standard_normal((3, n, n)) + 1j * rng.standard_normal((3, n, n))).astype(np.complex64)
    fwd = A.fft2d(torch.from_numpy(x).cuda()).cpu().numpy()
    inv = A.fft2d(torch.from_numpy(x).cuda(), inverse=True).cpu().numpy()
    for b in range(3):
        assert rel_l2(fwd[b] / (n * n), O.fft2n(x[b].astype(np.complex128))) < 5e-7
        assert rel_l2(inv[b], O.ifft2u(x[b].astype(np.complex128))) < 5e-7
    if n == 64:     # and against the definition of the DFT itself
        assert rel_l2(fwd[0], O.naive_dft2(x[0].astype(np.complex128))) < 5e-7


# ---------------------------------------------------------------------------------- configs 0, 1

@pytest.mark.parametrize("mx,my", [(96, 160), (160, 128), (192, 96), (128, 256), (256, 192)])
def test_reduced_grid_line_transforms(A, mx, my):
    """fft_xy.cuh (lengths 16*R1, R1 in {6,8,10,12,16}) against the DFT: type X alone as a 2-D
    transform (forward and inverse), and X followed by Y as the identity."""
    import torch
    rng = np.random.default_rng(mx * 1000 + my)
    x = (rng.standard_normal((3, my, mx)) + 1j * rng.standard_normal((3, my, mx))).astype(np.complex64)
    for mode in (0, 1):
        y = A.fft2d_xy(torch.from_numpy(x.copy()).cuda(), mode).cpu().numpy()
        ref = np.fft.fft2(x.astype(np.complex128)) if mode == 0 else np.fft.ifft2(x.astype(np.complex128)) * (mx * my)
        assert rel_l2(y, ref) < 2e-6, (mx, my, mode)
    for mode in (2, 3):
        y = A.fft2d_xy(torch.from_numpy(x.copy()).cuda(), mode).cpu().numpy()
        assert rel_l2(y, x) < 2e-6, (mx, my, mode)


@pytest.mark.parametrize("index", [0, 1])
def test_single_tile_configs(A, index):
    cfg = get_config(index)
    stacks, _ = make_batch(cfg, [0])
    refs, geo = oracle_reconstruct(cfg, stacks)
    plan, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks)
    check_tile(refs[0], field[0], zern[0], pupil[0], status[0], cfg.name)
    # stage level: sub-spectra on the discs (Eq. 7) and the stitched spectrum
    S = plan.debug_buffer(A.DBG_SUBSPECTRA, 1).cpu().numpy()[0]
    s_ref = np.concatenate([refs[0].spectra[i][geo.disc_b[i]] for i in range(cfg.n_bright)])
    assert rel_l2(S, s_ref) < 1e-5
    Og = plan.debug_buffer(A.DBG_OBJECT_SPECTRUM, 1).cpu().numpy()[0].reshape(cfg.tile_n, cfg.tile_n)
    assert rel_l2(Og, np.fft.ifftshift(refs[0].o_hat)) < 1e-5
    assert np.array_equal(Og != 0, np.fft.ifftshift(refs[0].known))


# ---------------------------------------------------------------------------------- config 2
@pytest.mark.parametrize("df_mode", [0, 1, 2])
def test_config2_reduced_all_tiles_ragged_chunks(A, df_mode):
    """64x64 variant of config 2 (8 + 16 LEDs, Poisson noise, 3x grid): every tile against the
    oracle, with 5 tiles over chunks of 2 (two full chunks and a ragged tail); both darkfield
    schedulers (persistent task kernel / one launch per phase)."""
    cfg = get_config(2, tile_n=64, batch=5, grid=(3, 2))
    stacks, _ = make_batch(cfg, range(5))
    refs, _ = oracle_reconstruct(cfg, stacks)
    plan, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks, chunk_tiles=2, df_mode=df_mode)
    assert plan.info["chunk_tiles"] == 2
    for b in range(5):
        check_tile(refs[b], field[b], zern[b], pupil[b], status[b], f"cfg2@64 tile {b}")
    its = plan.debug_buffer(A.DBG_DF_ITERS, 1).cpu().numpy()
    assert its.min() >= 1 and its.max() < 48          # CG converged by its tolerance, not the cap


@pytest.mark.parametrize("df_mode", [0, 1, 2])
def test_config2_128(A, df_mode):
    cfg = get_config(2, tile_n=128, batch=3, grid=(2, 2))
    stacks, _ = make_batch(cfg, range(3))
    refs, _ = oracle_reconstruct(cfg, stacks)
    _, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks, df_mode=df_mode)
    for b in range(3):
        check_tile(refs[b], field[b], zern[b], pupil[b], status[b], f"cfg2@128 tile {b}")


def test_config2_full_size_bench_configuration(A):
    """Config 2 at full size in the launch configuration bench.py times (batch 64, default chunk):
    sampled tiles against the oracle, properties on every tile."""
    cfg = get_config(2)
    tiles = list(range(64))
    stacks, truths = make_batch(cfg, tiles)
    plan, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks)
    assert np.all(status == 0)
    # the same batch in three balanced internal passes (22 + 21 + 21 tiles) gives the same bits
    _, field3, zern3, _, _ = gpu_reconstruct(A, cfg, stacks, chunk_tiles=24)
    assert np.array_equal(field, field3) and np.array_equal(zern, zern3)
    # the darkfield solver on the full N x N grid (df_mode 3) solves the same least-squares problems as the
    # default reduced cyclic grids: both stop at the same CG tolerance, so they agree far inside the parity bar
    _, field_full, zern_full, _, _ = gpu_reconstruct(A, cfg, stacks[:8], df_mode=3)
    assert np.array_equal(zern_full, zern[:8])
    for b in range(8):
        assert rel_l2(field[b], field_full[b]) < 2e-5, b
    sample = [0, 37, 63]
    refs, _ = oracle_reconstruct(cfg, stacks[sample])
    for ref, b in zip(refs, sample):
        check_tile(ref, field[b], zern[b], pupil[b], status[b], f"cfg2 tile {b}")
    # properties that hold for every tile: DC real-positive (R14); recovered coefficients close
    # to the injected ones (BASELINE.json: < 1e-3 rad RMS under this noise)
    for b in tiles:
        dc = field[b].mean()
        assert dc.real > 0 and abs(dc.imag) < 1e-4 * abs(dc)
        ct = np.array([truths[b].coef[j] for j in cfg.noll_fit])
        assert np.linalg.norm(zern[b] - ct) < 1e-3, f"tile {b}"


# ---------------------------------------------------------------------------------- config 3
def test_config3_256_all_leds(A):
    """Config 3's optics (12 + 32 LEDs on three rings, 34 fitted Zernike terms) at N = 256 with the
    pupil strength scaled to stay inside the validity bound of the re-wrapped fit (R11)."""
    cfg = get_config(3, tile_n=256, batch=1, pupil_strength=0.5)
    stacks, _ = make_batch(cfg, [0])
    refs, _ = oracle_reconstruct(cfg, stacks)
    _, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks)
    check_tile(refs[0], field[0], zern[0], pupil[0], status[0], "cfg3@256")


def test_config3_full_tile_size_first_ring(A):
    """N = 512, u = 3 (the largest kernels: 3-pass FFT, 1536^2 output), 12 NA-matching LEDs,
    34 terms at the config's 1 rad RMS, darkfield restricted to the first ring so that the dense
    fp64 oracle finishes in about two minutes."""
    cfg = get_config(3, batch=2, dark_rings=((0.28, 8),))
    stacks, _ = make_batch(cfg, [0, 1])
    refs, _ = oracle_reconstruct(cfg, stacks[:1])
    _, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks)
    check_tile(refs[0], field[0], zern[0], pupil[0], status[0], "cfg3@512 ring0")
    assert status[1] == 0


# ---------------------------------------------------------------------------------- config 4 features
def test_background_skip_bad_input_and_compaction(A):
    """Config 4's structure at 64x64: blank tiles (amp 1, phase 0) must come back with status 1 and
    zero outputs (R18), a tile with a NaN pixel with status 2, and the
    remaining tiles, compacted into ragged chunks, must match the oracle."""
    cfg = get_config(4, tile_n=64, batch=11, grid=(4, 3))
    blank = np.array([0, 1, 0, 0, 1, 1, 0, 1, 0, 0, 1], dtype=bool)
    stacks = np.empty((11, cfg.n_bright + cfg.n_dark, 64, 64), np.float32)
    from apic_synth import make_tile
    for t in range(11):
        stacks[t], _ = make_tile(cfg, t, blank=bool(blank[t]))
    stacks[6, 3, 5, 7] = np.nan
    kw = dict(bg_mode=1, bg_threshold=0.9)
    p = oracle_params(cfg, **kw)
    refs = O.reconstruct_batch(stacks, p)
    plan, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks, chunk_tiles=4, **kw)
    expect = np.array([r.status for r in refs])
    assert np.array_equal(status, expect)
    assert np.array_equal(expect == 1, blank) and expect[6] == 2
    for b in range(11):
        if expect[b] in (1, 2):
            assert not field[b].any() and not zern[b].any() and not pupil[b].any()
        else:
            check_tile(refs[b], field[b], zern[b], pupil[b], status[b], f"cfg4@64 tile {b}")


def test_variance_background_mode_matches_oracle(A):
    cfg = get_config(4, tile_n=64, batch=4, grid=(2, 2))
    from apic_synth import make_tile
    stacks = np.stack([make_tile(cfg, t, blank=(t % 2 == 1))[0] for t in range(4)])
    kw = dict(bg_mode=2, bg_threshold=1e-2)
    refs = O.reconstruct_batch(stacks, oracle_params(cfg, **kw))
    _, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks, **kw)
    assert status.tolist() == [r.status for r in refs] == [0, 1, 0, 1]


def test_all_tiles_background_is_a_no_op(A):
    cfg = get_config(4, tile_n=64, batch=3, grid=(2, 2))
    from apic_synth import make_tile
    stacks = np.stack([make_tile(cfg, t, blank=True)[0] for t in range(3)])
    _, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks, bg_mode=1, bg_threshold=0.9)
    assert status.tolist() == [1, 1, 1] and not field.any()


# ---------------------------------------------------------------------------------- misc contract
def test_results_are_bit_reproducible_and_batch_invariant(A):
    """No atomics on the data path: two runs are bit-identical, and a tile's result does not depend
    on its position in the batch or on the chunking."""
    cfg = get_config(2, tile_n=64, batch=4, grid=(2, 2))
    stacks, _ = make_batch(cfg, range(4))
    _, f1, z1, _, _ = gpu_reconstruct(A, cfg, stacks)
    _, f2, z2, _, _ = gpu_reconstruct(A, cfg, stacks)
    assert np.array_equal(f1, f2) and np.array_equal(z1, z2)
    _, f3, z3, _, _ = gpu_reconstruct(A, cfg, stacks[::-1].copy(), chunk_tiles=3)
    assert np.array_equal(f1, f3[::-1]) and np.array_equal(z1, z3[::-1])
    for team in (1, 2, 4):                                            # team size does not change the arithmetic
        _, ft, zt, _, _ = gpu_reconstruct(A, cfg, stacks, df_team=team)
        assert np.array_equal(f1, ft) and np.array_equal(z1, zt), team
    _, f4, z4, _, _ = gpu_reconstruct(A, cfg, stacks, df_mode=1)      # the launch-per-phase and the ticket
    _, f5, z5, _, _ = gpu_reconstruct(A, cfg, stacks, df_mode=2)      # schedulers share their task bodies
    assert np.array_equal(f4, f5) and np.array_equal(z4, z5)
    # the team kernel sums the CG dot products in a different order: same result within fp32 rounding
    assert np.linalg.norm(f1 - f4) <= 1e-5 * np.linalg.norm(f4) and np.array_equal(z1, z4)


def test_host_entry_point_and_batch_limits(A):
    import torch
    cfg = get_config(0)
    stacks, _ = make_batch(cfg, [0])
    plan = A.Plan.from_config(cfg, max_batch=2)
    x = torch.from_numpy(stacks).cuda()
    field, zern, pupil, status = plan.reconstruct(x)
    n, on = cfg.tile_n, cfg.out_n
    h_field = np.empty((1, on, on), np.complex64)
    h_zern = np.empty((1, plan.nz), np.float32)
    h_pupil = np.empty((1, n, n), np.complex64)
    h_status = np.empty((1,), np.int32)
    plan.reconstruct_host(stacks, h_field, h_zern, h_pupil, h_status)
    assert np.array_equal(h_field, field.cpu().numpy()) and np.array_equal(h_zern, zern.cpu().numpy())
    assert np.array_equal(h_pupil, pupil.cpu().numpy()) and h_status[0] == 0
    big = torch.zeros((3, cfg.n_bright, n, n), device="cuda")
    with pytest.raises(A.ApicError, match="batch"):
        plan.reconstruct(big)
    assert plan.last_launch_count > 0


def test_uint16_entry_equals_fp32_entry_on_the_same_values(A):
    """apic_reconstruct_u16 (raw counts + per-image scale, conversion fused into the S0 pass) must give
    the fp32 entry's bits on float(count) * scale, through the device and the host entry points; a
    non-finite scale is bad input."""
    import torch
    cfg = get_config(2, tile_n=64, batch=4, grid=(2, 2))
    stacks, truths = make_batch(cfg, [0, 1, 2, 3])
    nb = cfg.n_bright
    gains = np.array([[t.gain_bright] * nb + [t.gain_dark] * cfg.n_dark for t in truths])        # photons per unit
    raw = np.rint(stacks.astype(np.float64) * gains[:, :, None, None])
    assert raw.min() >= 0 and raw.max() <= 65535
    raw = raw.astype(np.uint16)
    scale = (1.0 / gains).astype(np.float32)
    x32 = raw.astype(np.float32) * scale[:, :, None, None]                                          # fp32 product
    assert np.allclose(x32, stacks, rtol=1e-6)
    plan = A.Plan.from_config(cfg, max_batch=4)
    ref = [o.cpu().numpy() for o in plan.reconstruct(torch.from_numpy(x32).cuda())]
    got = [o.cpu().numpy() for o in plan.reconstruct_u16(torch.from_numpy(raw).cuda(), torch.from_numpy(scale).cuda())]
    for a, b in zip(ref, got):
        assert np.array_equal(a, b)
    assert np.all(ref[3] == 0)
    # host entry
    field = np.empty_like(ref[0]); zern = np.empty_like(ref[1]); pupil = np.empty_like(ref[2]); status = np.empty_like(ref[3])
    plan.reconstruct_host_u16(raw, scale, field, zern, pupil, status)
    assert np.array_equal(field, ref[0]) and np.array_equal(zern, ref[1]) and np.array_equal(status, ref[3])
    # a non-finite scale flags the tile and leaves the others untouched
    bad = scale.copy()
    bad[2, 5] = np.inf
    got = [o.cpu().numpy() for o in plan.reconstruct_u16(torch.from_numpy(raw).cuda(), torch.from_numpy(bad).cuda())]
    assert list(got[3]) == [0, 0, 2, 0] and np.all(got[0][2] == 0)
    assert np.array_equal(got[0][[0, 1, 3]], ref[0][[0, 1, 3]])


def test_host_entry_pipelines_sub_batches_without_changing_bits(A):
    """apic_reconstruct_host splits batches of >= 64 tiles into sub-batches whose uploads / kernels /
    downloads overlap on separate streams: same bits as one device call on the whole batch."""
    import torch
    cfg = get_config(2, tile_n=64, batch=4, grid=(2, 2))
    stacks, _ = make_batch(cfg, [0, 1, 2, 3])
    big = np.ascontiguousarray(np.concatenate([stacks] * 18)[:70])
    plan = A.Plan.from_config(cfg, max_batch=70)
    ref = [o.cpu().numpy() for o in plan.reconstruct(torch.from_numpy(big).cuda())]
    field = np.empty_like(ref[0]); zern = np.empty_like(ref[1]); pupil = np.empty_like(ref[2]); status = np.empty_like(ref[3])
    for _ in range(2):
        field[:] = 0
        plan.reconstruct_host(big, field, zern, pupil, status)
        assert np.array_equal(field, ref[0]) and np.array_equal(zern, ref[1])
        assert np.array_equal(pupil, ref[2]) and np.array_equal(status, ref[3])
    assert np.array_equal(field[0], field[4]) and np.array_equal(field[1], field[69])


def test_config4_full_tile_size_with_background_tiles(A):
    """Config 4's tiles at full size (256 x 256, 8 + 16 LEDs, the reduced-grid darkfield kernel) with
    blank tiles in the batch: statuses of every tile, zero outputs for the skipped ones, one live tile
    against the oracle, and the live tiles independent of the blank ones around them."""
    from apic_synth import make_tile
    cfg = get_config(4, batch=7, grid=(4, 2))
    blank = np.array([1, 0, 1, 0, 0, 1, 0], dtype=bool)
    stacks = np.empty((7, cfg.n_bright + cfg.n_dark, cfg.tile_n, cfg.tile_n), np.float32)
    for t in range(7):
        stacks[t], _ = make_tile(cfg, t, blank=bool(blank[t]))
    kw = dict(bg_mode=1, bg_threshold=0.9)
    plan, field, zern, pupil, status = gpu_reconstruct(A, cfg, stacks, chunk_tiles=3, **kw)
    assert np.array_equal(status == 1, blank) and np.all(status[~blank] == 0)
    for b in np.nonzero(blank)[0]:
        assert not field[b].any() and not zern[b].any() and not pupil[b].any()
    p = oracle_params(cfg, **kw)
    ref = O.reconstruct_tile(stacks[3], p)
    check_tile(ref, field[3], zern[3], pupil[3], status[3], "cfg4 tile 3")
    _, field1, zern1, _, status1 = gpu_reconstruct(A, cfg, stacks[[1, 3, 4, 6]], **kw)
    assert np.array_equal(field1, field[[1, 3, 4, 6]]) and np.array_equal(zern1, zern[[1, 3, 4, 6]])
