"""ORACLE of the consumer-facing outputs built from the event stream.  TEST INFRASTRUCTURE ONLY.

Plain numpy in float64, written from the paper's text; shares nothing with the CUDA path.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.

voxel_grid -- PAPER.md:331 (Supp. C, "Training Details"): "Each 0.5 s event segment is represented as a
    per-polarity event voxel grid discretized into 128 temporal bins with linear interpolation applied along
    the time axis.  Each bin is normalized by dividing by its maximum event count."  ("A
    per-polarity, 128-bin event voxel (256 channels)"; "10 ms event accumulations".)
    Reading R30: a window of duration D starting at t0 and B bins; bin centres sit at
    tau = 0 .. B-1 with tau = (B - 1) (t - t0) / D, and an event adds max(0, 1 - |tau - b|) to bin b of its
    pixel in the channel of its polarity (ON = 0, OFF = 1) -- the two bins that bracket tau share one unit,
    so an event always adds exactly 1 in total and B = 1 is the plain per-polarity accumulation image.
    "Normalized": every (env, polarity, bin) plane divided by its own maximum when that is > 0.

sort_by_time -- the time-sorted per-environment stream (the stream E = {(u_k, t_k, p_k)}):
    events ordered by (env, t, y, x, polarity-independent crossing order k); the definition is a stable sort.
"""
from __future__ import annotations

import numpy as np


def voxel_grid(env, x, y, p, t, num_envs: int, height: int, width: int, bins: int, t0: float, duration: float,
               normalize: bool = False) -> np.ndarray:
    """Events (arrays of equal length: env, x, y, polarity +1/-1, absolute time t in seconds) ->
    V [E, 2, B, H, W] float64.  Events outside [t0, t0 + duration] are ignored."""
    env = np.asarray(env, np.int64); x = np.asarray(x, np.int64); y = np.asarray(y, np.int64)
    p = np.asarray(p, np.int64); t = np.asarray(t, np.float64)
    V = np.zeros((num_envs, 2, bins, height, width), np.float64)
    keep = (t >= t0) & (t <= t0 + duration)
    env, x, y, p, t = env[keep], x[keep], y[keep], p[keep], t[keep]
    tau = (bins - 1) * (t - t0) / duration
    ch = np.where(p > 0, 0, 1)
    for b in range(bins):
        w = np.maximum(0.0, 1.0 - np.abs(tau - b))
        np.add.at(V, (env, ch, b, y, x), w)
    if normalize:
        m = V.max(axis=(3, 4), keepdims=True)
        V = np.where(m > 0, V / np.where(m > 0, m, 1.0), V)
    return V


def sort_by_time(env, t, y, x, k):
    """Index array that puts the events in (env, t, y, x, k) order."""
    return np.lexsort((np.asarray(k), np.asarray(x), np.asarray(y), np.asarray(t), np.asarray(env)))
