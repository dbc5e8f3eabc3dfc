"""GPU parity of apic_reassemble (within-FOV reassembly) against
oracle/reassemble_oracle.py, element by element on the same seeded inputs, through the C ABI.  fp32 against fp64:
the blend is <= 4 products per pixel, so 2e-6 relative is the arithmetic's bound; the unit factors come from fp64
accumulations of exact fp32 products on both sides, so they agree to fp32 rounding of the output (1e-6)."""
import numpy as np
import pytest

from oracle import reassemble_oracle as R

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def A():
    import torch
    assert torch.cuda.is_available()
    import paper_2407_20469_b200 as pkg
    pkg.load()
    return pkg


def _tiles(seed, ty, tx, t, blank=()):
    rng = np.random.default_rng(seed)
    amp = 0.6 + 0.4 * rng.random((ty, tx, t, t))
    f = (amp * np.exp(1j * rng.uniform(-np.pi, np.pi, (ty, tx, t, t)))).astype(np.complex64)
    for rc in blank:
        f[rc] = 0
    return f


def _run(A, f, ov, align):
    import torch
    fov, u = A.reassemble(torch.from_numpy(f).cuda(), ov, align)
    torch.cuda.synchronize()
    return fov.cpu().numpy(), u.cpu().numpy()


@pytest.mark.parametrize("ty,tx,t,ov,align", [(1, 1, 64, 6, True), (3, 4, 96, 10, True), (3, 4, 96, 10, False),
                                                (2, 5, 50, 25, True), (4, 3, 33, 0, True), (5, 5, 768, 76, True)])
def test_reassembly_matches_the_oracle(A, ty, tx, t, ov, align):
    f = _tiles(10 * ty + tx + ov, ty, tx, t)
    # overlapping content must be consistent for the alignment to be meaningful: cut the tiles from one FOV and give
    # every tile its own global phase, as apic_reconstruct does (DC real-positive per tile)
    h, w = R.fov_size(ty, t, ov), R.fov_size(tx, t, ov)
    big = _tiles(99, 1, 1, max(h, w))[0, 0][:h, :w]
    step = t - ov
    rng = np.random.default_rng(5)
    for r in range(ty):
        for c in range(tx):
            f[r, c] = big[r * step:r * step + t, c * step:c * step + t] * np.exp(1j * rng.uniform(-np.pi, np.pi))
    f = f.astype(np.complex64)
    fov, u = _run(A, f, ov, align)
    ref, uref = R.reassemble(f, ov, align)
    assert fov.shape == ref.shape
    assert np.abs(u - uref).max() < 1e-6
    assert np.abs(fov - ref).max() <= 2e-6 * np.abs(ref).max()
    if align and ov > 0:
        # and it is the FOV the tiles were cut from, at the phase of tile (0, 0)
        ph = f[0, 0, 0, 0] / big[0, 0]
        assert np.abs(fov - big * ph).max() < 5e-6


def test_unrelated_and_blank_tiles(A):
    """Random unrelated tiles (the factors are then arbitrary but must equal the oracle's), blank tiles (factor 1)."""
    f = _tiles(3, 3, 3, 40, blank=[(1, 1), (2, 0)])
    fov, u = _run(A, f, 8, True)
    ref, uref = R.reassemble(f, 8, True)
    assert np.abs(u - uref).max() < 1e-5 and np.abs(fov - ref).max() <= 2e-5 * np.abs(ref).max()
    z = np.zeros((2, 2, 16, 16), dtype=np.complex64)
    fov, u = _run(A, z, 4, True)
    assert not fov.any() and np.array_equal(u, np.ones((2, 2), dtype=np.complex64))


def test_bad_geometry_is_rejected(A):
    import torch
    f = torch.zeros((2, 2, 16, 16), dtype=torch.complex64, device="cuda")
    with pytest.raises(A.ApicError):
        A.reassemble(f, 9)                       # 2 overlap > T
    with pytest.raises(A.ApicError):
        A.reassemble(f.to(torch.complex128), 2)


def test_reconstructed_tiles_of_one_field_reassemble_without_seams(A):
    """End to end: four overlapping 64 x 64 windows of ONE periodic synthetic object are reconstructed independently
    (config 0 optics: each comes out with its own DC real-positive) and reassembled; after alignment the two
    reconstructions of every overlap pixel agree, without it they differ by the tiles' global phases."""
    import torch
    from apic_synth import get_config, make_tile, plan_args
    cfg = get_config(0)
    stack, truth = make_tile(cfg, 0)
    n, up = cfg.tile_n, cfg.upsample
    plan = A.Plan(*plan_args(cfg), max_batch=4)
    # the object is periodic on the tile, so a cyclic shift of the stack is another valid tile of the same object
    sh = n // 2
    stacks = np.stack([stack, np.roll(stack, -sh, axis=2), np.roll(stack, -sh, axis=1), np.roll(stack, (-sh, -sh), axis=(1, 2))])
    field, zern, pupil, status = plan.reconstruct(torch.from_numpy(stacks).cuda())
    assert status.cpu().numpy().tolist() == [0, 0, 0, 0]
    t, ov = n * up, (n - sh) * up
    f = field.reshape(2, 2, t, t).contiguous()
    fov, u = A.reassemble(f, ov, True)
    fov0, _ = A.reassemble(f, ov, False)
    torch.cuda.synchronize()
    ref, uref = R.reassemble(f.cpu().numpy(), ov, True)
    assert np.abs(fov.cpu().numpy() - ref).max() <= 5e-6 * np.abs(ref).max()
    # the reassembled FOV equals tile (0, 0)'s own reconstruction continued periodically
    f00 = f[0, 0].cpu().numpy()
    ext = np.tile(f00, (2, 2))[:fov.shape[0], :fov.shape[1]]
    assert np.abs(fov.cpu().numpy() - ext).max() < 2e-3 * np.abs(ext).max()
