"""Pins of oracle/reassemble_oracle.py (within-FOV reassembly; readings B6-B8).
None of the expected values comes from the oracle itself: a hand-computed ramp, a ground-truth FOV the tiles are cut
from, plain tiling, and a brute-force per-pixel evaluation written straight from the definition."""
import numpy as np
import pytest

from oracle import reassemble_oracle as R


def _cut(fov, ty, tx, t, ov):
    step = t - ov
    return np.array([[fov[r * step:r * step + t, c * step:c * step + t] for c in range(tx)] for r in range(ty)])


def _random_fov(rng, h, w):
    amp = 0.6 + 0.4 * rng.random((h, w))
    return amp * np.exp(1j * rng.uniform(-np.pi, np.pi, (h, w)))


def test_ramp_by_hand():
    # overlap 4: the rising tile weighs 1/8, 3/8, 5/8, 7/8; the falling one the complement
    w_mid = R.ramp_weights(10, 4, first=False, last=False)
    assert np.allclose(w_mid, [0.125, 0.375, 0.625, 0.875, 1, 1, 0.875, 0.625, 0.375, 0.125], atol=0, rtol=0)
    assert np.array_equal(R.ramp_weights(10, 4, first=True, last=True), np.ones(10))
    assert np.array_equal(R.ramp_weights(6, 0, first=False, last=False), np.ones(6))
    assert R.fov_size(5, 768, 76) == 5 * 692 + 76


@pytest.mark.parametrize("ty,tx,t,ov", [(1, 1, 8, 2), (2, 3, 16, 4), (3, 2, 12, 6), (4, 4, 10, 1)])
def test_weights_are_a_partition_of_unity(ty, tx, t, ov):
    ones = np.ones((ty, tx, t, t), dtype=complex)
    fov, u = R.reassemble(ones, ov, align=False)
    assert np.abs(fov - 1.0).max() < 1e-15
    fov, u = R.reassemble(ones, ov, align=True)          # identical tiles: every factor is 1
    assert np.abs(u - 1.0).max() < 1e-15 and np.abs(fov - 1.0).max() < 1e-15


@pytest.mark.parametrize("ty,tx,t,ov", [(2, 2, 16, 4), (3, 4, 24, 6), (5, 5, 20, 2)])
def test_tiles_cut_from_a_fov_reassemble_to_it_whatever_their_global_phases(ty, tx, t, ov):
    rng = np.random.default_rng(100 * ty + tx)
    truth = _random_fov(rng, R.fov_size(ty, t, ov), R.fov_size(tx, t, ov))
    tiles = _cut(truth, ty, tx, t, ov)
    plain, _ = R.reassemble(tiles, ov, align=False)
    assert np.abs(plain - truth).max() < 1e-13
    factors = np.exp(1j * rng.uniform(-np.pi, np.pi, (ty, tx)))
    fov, u = R.reassemble(tiles * factors[:, :, None, None], ov, align=True)
    # everything is brought to the phase of tile (0, 0)
    assert np.abs(fov - truth * factors[0, 0]).max() < 1e-12
    assert np.abs(u * factors - factors[0, 0]).max() < 1e-12
    # without alignment the seams do not match: the test above is not vacuous
    bad, _ = R.reassemble(tiles * factors[:, :, None, None], ov, align=False)
    assert np.abs(bad - truth * factors[0, 0]).max() > 0.1


def test_overlap_zero_is_plain_tiling_and_blank_overlaps_keep_unit_factors():
    rng = np.random.default_rng(7)
    tiles = _random_fov(rng, 6 * 8, 8).reshape(2, 3, 8, 8)
    fov, u = R.reassemble(tiles, 0, align=True)
    assert np.array_equal(u, np.ones((2, 3)))
    for r in range(2):
        for c in range(3):
            assert np.array_equal(fov[r * 8:(r + 1) * 8, c * 8:(c + 1) * 8], tiles[r, c])
    blank = np.zeros((2, 2, 8, 8), dtype=complex)
    fov, u = R.reassemble(blank, 2, align=True)
    assert np.array_equal(u, np.ones((2, 2))) and not fov.any()


def test_against_a_per_pixel_evaluation_of_the_definition():
    """B6-B8 written out pixel by pixel (no slicing, no outer products) on a tiny case."""
    rng = np.random.default_rng(11)
    ty, tx, t, ov = 3, 2, 6, 2
    tiles = _random_fov(rng, ty * tx * t, t).reshape(ty, tx, t, t)
    fov, u = R.reassemble(tiles, ov, align=True)
    step = t - ov
    # factors from the definition
    uu = np.ones((ty, tx), dtype=complex)
    for r in range(ty):
        for c in range(tx):
            if r == 0 and c == 0:
                continue
            acc = 0j
            if c > 0:
                for y in range(t):
                    for k in range(ov):
                        acc += uu[r, c - 1] * tiles[r, c - 1, y, step + k] * np.conj(tiles[r, c, y, k])
            if r > 0:
                for k in range(ov):
                    for x in range(t):
                        acc += uu[r - 1, c] * tiles[r - 1, c, step + k, x] * np.conj(tiles[r, c, k, x])
            uu[r, c] = acc / abs(acc)
    assert np.abs(uu - u).max() < 1e-13

    def w1(i, idx, n):
        if idx > 0 and i < ov:
            return (i + 0.5) / ov
        if idx < n - 1 and i >= t - ov:
            return 1.0 - (i - (t - ov) + 0.5) / ov
        return 1.0
    for Y in range(fov.shape[0]):
        for X in range(fov.shape[1]):
            acc, wsum = 0j, 0.0
            for r in range(ty):
                for c in range(tx):
                    y, x = Y - r * step, X - c * step
                    if 0 <= y < t and 0 <= x < t:
                        w = w1(y, r, ty) * w1(x, c, tx)
                        acc += w * uu[r, c] * tiles[r, c, y, x]
                        wsum += w
            assert abs(wsum - 1.0) < 1e-14
            assert abs(acc - fov[Y, X]) < 1e-13
