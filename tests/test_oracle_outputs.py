"""Pins for oracle/evis_outputs.py (voxel grid, time-sorted stream): hand-worked values, library routines and
invariants -- never the oracle against itself.  CPU only."""
import os

import numpy as np

from oracle import evis_outputs as out

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_p17_voxel_grid_hand_worked():
    """tests/golden/voxel_by_hand.txt: six events of one pixel with weights worked out by hand from PAPER.md:331 /
    reading R30 (swapped bracket weights, a B instead of B - 1 scale, or swapped polarity channels all fail)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "voxel_by_hand.txt")) if l.strip() and not l.startswith("#")]
    want = np.zeros((2, 5))
    for r in rows:
        want[int(r[0])] = [float(v) for v in r[1:]]
    t = np.array([2.00, 2.25, 2.30, 2.55, 2.95, 3.00, 3.10])
    p = np.array([+1, +1, -1, +1, -1, +1, +1])
    z = np.zeros(len(t), np.int64)
    V = out.voxel_grid(z, z + 2, z + 1, p, t, num_envs=1, height=3, width=4, bins=5, t0=2.0, duration=1.0)
    assert V.shape == (1, 2, 5, 3, 4)
    assert np.allclose(V[0, :, :, 1, 2], want, atol=1e-12)
    V[0, :, :, 1, 2] = 0
    assert not V.any()                                # nothing lands on another pixel


def test_p17b_one_bin_is_the_accumulation_image():
    """B = 1 ('10 ms event accumulations'): the grid is the per-polarity event count of every pixel,
    checked against np.bincount on the flattened (env, channel, y, x) index."""
    rng = np.random.default_rng(5)
    n, E, H, W = 5000, 3, 7, 9
    env, x, y = rng.integers(0, E, n), rng.integers(0, W, n), rng.integers(0, H, n)
    p = rng.choice([-1, 1], n)
    t = rng.uniform(0.0, 0.01, n)
    V = out.voxel_grid(env, x, y, p, t, E, H, W, bins=1, t0=0.0, duration=0.01)
    flat = ((env * 2 + (p < 0)) * H + y) * W + x
    assert np.array_equal(V.reshape(-1), np.bincount(flat, minlength=E * 2 * H * W).astype(np.float64))


def test_p17c_voxel_grid_preserves_count_and_mean_time():
    """Linear interpolation along time splits one unit between the two bracketing bins: per pixel and polarity the
    bins sum to the event count, and sum_b b V[b] equals the sum of tau = (B - 1)(t - t0) / D over the events."""
    rng = np.random.default_rng(6)
    n, E, H, W, B = 4000, 2, 5, 6, 16
    env, x, y = rng.integers(0, E, n), rng.integers(0, W, n), rng.integers(0, H, n)
    p = rng.choice([-1, 1], n)
    t0, D = 1.5, 0.25
    t = rng.uniform(t0, t0 + D, n)
    V = out.voxel_grid(env, x, y, p, t, E, H, W, bins=B, t0=t0, duration=D)
    cnt = np.zeros((E, 2, H, W)); mom = np.zeros((E, 2, H, W))
    np.add.at(cnt, (env, (p < 0).astype(int), y, x), 1.0)
    np.add.at(mom, (env, (p < 0).astype(int), y, x), (B - 1) * (t - t0) / D)
    assert np.allclose(V.sum(axis=2), cnt, atol=1e-9)
    assert np.allclose((V * np.arange(B)[None, None, :, None, None]).sum(axis=2), mom, atol=1e-9)
    assert V.min() >= 0.0


def test_p17d_normalized_planes():
    """'Each bin is normalized by dividing by its maximum event count': every non-empty (env, polarity,
    bin) plane has maximum 1 and keeps its ratios; empty planes stay zero."""
    rng = np.random.default_rng(7)
    n, E, H, W, B = 3000, 2, 4, 5, 4
    env, x, y = rng.integers(0, E, n), rng.integers(0, W, n), rng.integers(0, H, n)
    p = np.where(env == 0, 1, rng.choice([-1, 1], n))          # env 0 has no OFF events at all
    t = rng.uniform(0.0, 1.0, n)
    V = out.voxel_grid(env, x, y, p, t, E, H, W, B, 0.0, 1.0)
    N = out.voxel_grid(env, x, y, p, t, E, H, W, B, 0.0, 1.0, normalize=True)
    m = V.max(axis=(3, 4))
    assert not N[0, 1].any() and not V[0, 1].any()
    assert np.allclose(N.max(axis=(3, 4))[m > 0], 1.0)
    assert np.allclose(N * m[..., None, None], V, atol=1e-12)


def test_p18_time_sorted_stream_is_a_stable_sort():
    """The time-sorted per-env stream: envs ascending, times non-decreasing inside an env, a permutation of
    the input, ties kept in (y, x, k) order."""
    rng = np.random.default_rng(8)
    n = 2000
    env, x, y, k = rng.integers(0, 4, n), rng.integers(0, 9, n), rng.integers(0, 7, n), rng.integers(1, 4, n)
    t = np.round(rng.uniform(0, 1e-2, n), 4)                   # many equal stamps
    o = out.sort_by_time(env, t, y, x, k)
    assert np.array_equal(np.sort(o), np.arange(n))
    key = np.stack([env[o], t[o], y[o], x[o], k[o]], axis=1)
    d = np.diff(key, axis=0)
    first = np.argmax(d != 0, axis=1)
    assert np.all(d[np.arange(n - 1), first] >= 0)
