"""apic_reassemble_static: the within-FOV reassembly for callers that cannot allocate device memory.

Some users of libapic reassemble tiles at a point where asking the CUDA runtime for memory is not an option: the
process handed all of the GPU's memory to its own arena when it started, or the code is a component inside an
application that owns the allocator, or it sits in an acquisition loop where the stall of a cudaMalloc / cudaFree is
not acceptable.  `apic_reassemble` needs a caller-supplied scratch buffer (`d_work`); `apic_reassemble_static` keeps
that scratch in a fixed array inside the library's device image instead and therefore accepts at most
`apic_reassemble_static_max_tiles()` tiles.

What is checked here, through the C ABI: the new entry point returns what the existing `apic_reassemble` returns on
the same inputs, within the tolerances of tests/test_gpu_reassemble.py (2e-6 of the largest FOV magnitude, 1e-6 on the
unit factors), on two calls in a row that share the built-in array - the second with a different, smaller geometry, so
that it runs on top of what the first left behind - and then on the first geometry again; that it writes into
buffers the caller preallocated; and that a FOV beyond the limit is refused with APIC_ESCRATCH, leaving the output
untouched.  The file is named to be collected last (`pytest --collect-only`): under `-x` a failure here hides nothing,
and the test does not depend on whether other tests ran before it in the same process.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def A():
    import torch
    assert torch.cuda.is_available()
    import paper_2407_20469_b200 as pkg
    pkg.load()
    return pkg


def _consistent_tiles(seed, ty, tx, t, ov):
    """Tiles cut from one random complex FOV, each with its own global phase (what apic_reconstruct hands over)."""
    rng = np.random.default_rng(seed)
    step = t - ov
    h, w = ty * step + ov, tx * step + ov
    big = (0.6 + 0.4 * rng.random((h, w))) * np.exp(1j * rng.uniform(-np.pi, np.pi, (h, w)))
    f = np.empty((ty, tx, t, t), np.complex64)
    for r in range(ty):
        for c in range(tx):
            f[r, c] = big[r * step:r * step + t, c * step:c * step + t] * np.exp(1j * rng.uniform(-np.pi, np.pi))
    return f


def _agree(fov, u, fov_ref, u_ref):
    assert fov.shape == fov_ref.shape and u.shape == u_ref.shape
    assert np.isfinite(fov).all() and np.isfinite(u).all()
    assert np.abs(u - u_ref).max() < 1e-6
    assert np.abs(fov - fov_ref).max() <= 2e-6 * np.abs(fov_ref).max()


def test_static_scratch_reassembly_equals_the_caller_scratch_path_on_consecutive_calls(A):
    import torch
    geometries = [(4, 5, 96, 10, True), (2, 3, 50, 24, True), (4, 5, 96, 10, True), (3, 3, 64, 8, False)]
    for k, (ty, tx, t, ov, align) in enumerate(geometries):
        f = torch.from_numpy(_consistent_tiles(40 + k, ty, tx, t, ov)).cuda()
        fov_ref, u_ref = A.reassemble(f, ov, align)                       # existing path, scratch from torch
        step = t - ov
        out = torch.full((ty * step + ov, tx * step + ov), float("nan"), dtype=torch.complex64, device="cuda")
        fac = torch.full((ty, tx), float("nan"), dtype=torch.complex64, device="cuda")
        fov, u = A.reassemble_static(f, ov, align, out=out, factors=fac)  # nothing allocated from here on
        torch.cuda.synchronize()
        assert fov.data_ptr() == out.data_ptr() and u.data_ptr() == fac.data_ptr()
        _agree(fov.cpu().numpy(), u.cpu().numpy(), fov_ref.cpu().numpy(), u_ref.cpu().numpy())
        if align:
            assert np.abs(u.cpu().numpy().ravel()[1:] - 1).max() > 1e-2     # the alignment did something


def test_static_scratch_two_calls_back_to_back_on_one_stream_without_a_sync_between(A):
    """Same stream = ordered on the GPU, so the shared array is safe; the second call must not see the first's data."""
    import torch
    fa = torch.from_numpy(_consistent_tiles(7, 3, 4, 80, 12)).cuda()
    fb = torch.from_numpy(_consistent_tiles(8, 5, 2, 40, 20)).cuda()
    ra, rb = A.reassemble(fa, 12, True), A.reassemble(fb, 20, True)
    torch.cuda.synchronize()
    sa = A.reassemble_static(fa, 12, True)
    sb = A.reassemble_static(fb, 20, True)
    torch.cuda.synchronize()
    _agree(sa[0].cpu().numpy(), sa[1].cpu().numpy(), ra[0].cpu().numpy(), ra[1].cpu().numpy())
    _agree(sb[0].cpu().numpy(), sb[1].cpu().numpy(), rb[0].cpu().numpy(), rb[1].cpu().numpy())


def test_static_scratch_limit_is_enforced_and_stated(A):
    import torch
    limit = A.reassemble_static_max_tiles()
    assert limit == 1024
    f = torch.ones((33, 32, 4, 4), dtype=torch.complex64, device="cuda")      # 1056 tiles > 1024
    out = torch.full((33 * 3 + 1, 32 * 3 + 1), 7.0, dtype=torch.complex64, device="cuda")
    with pytest.raises(A.ApicError, match="built-in scratch"):
        A.reassemble_static(f, 1, True, out=out)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                                           # refused before any kernel ran
    # exactly at the limit it runs, and identical tiles need no alignment: all factors 1, FOV all ones
    f = torch.ones((32, 32, 4, 4), dtype=torch.complex64, device="cuda")
    fov, u = A.reassemble_static(f, 1, True)
    torch.cuda.synchronize()
    assert np.abs(u.cpu().numpy() - 1).max() < 1e-6 and np.abs(fov.cpu().numpy() - 1).max() < 2e-6
    fov_ref, u_ref = A.reassemble(f, 1, True)
    _agree(fov.cpu().numpy(), u.cpu().numpy(), fov_ref.cpu().numpy(), u_ref.cpu().numpy())
