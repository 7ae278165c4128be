"""evis_voxelize_static -- the voxel grid for callers that may not allocate device memory.

Some users of this library run where cudaMalloc is forbidden: inside a rollout loop whose GPU memory the simulator, the
renderer and the learner divided among their own pools before the loop started (an allocation there can fail, and both
cudaMalloc and cudaFree hold up every stream of the device), or as a consumer of recorded events with no evis_ctx at all.
`Evis.set_voxels` allocates its accumulator, so it is closed to them; `evis_voxelize_static` builds the same grid from
finished events with its accumulator in a fixed 16 MiB array inside libevis.so.

The GPU test below checks that entry point against the existing path (evis_set_voxels / evis_read_voxels on the context
that produced the events) on TWO calls in a row with different shapes -- the array is shared between calls and keeps the
last call's contents, so the second call would show a missing clear.  Both paths run the same binary32 / fixed-point
arithmetic with integer sums, so the grids must be equal bit for bit (well inside the tolerance the voxel tests allow
against the oracle).  The file sorts last in the collection order on purpose (`pytest -x` stops at the first failure: a
failure here hides no other test), and the test makes no assumption about what ran before it: it passes alone in a
fresh process (its first call then does the one-time address look-up) and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2607_08098_b200 import binding, scenes


def test_limits_are_checked_without_a_gpu():
    """Sizes beyond the fixed accumulator are refused with EVIS_ERR_TOO_LARGE, bad arguments with INVALID_ARG, before any
    CUDA call (so this runs on a box without a GPU); the error text names the entry point."""
    L = binding.load()
    err = C.c_int(-1)
    fake = C.c_void_p(256)                      # never dereferenced: every call below fails validation first

    def call(n=0, E=1, H=8, W=8, bins=1, window=1, T=1 / 60, events=None, grid=fake):
        return L.evis_voxelize_static(events, n, E, H, W, bins, window, T, 0, 0, grid, None, C.byref(err))

    assert call(grid=None) == binding.EVIS_ERR_INVALID_ARG
    assert call(n=5) == binding.EVIS_ERR_INVALID_ARG                       # events missing
    for bad in (dict(E=0), dict(H=0), dict(W=-3), dict(bins=0), dict(window=0), dict(T=0.0), dict(T=float("nan")),
                dict(T=float("inf")), dict(E=70000), dict(H=40000)):
        assert call(**bad) == binding.EVIS_ERR_INVALID_ARG, bad
    # cfg 4's frame with 5 bins: two environments fit, three do not; neither do absurd sizes whose product wraps 2^64
    assert 2 * 2 * 5 * 260 * 346 <= binding.VOXELIZE_STATIC_MAX_CELLS < 2 * 3 * 5 * 260 * 346
    assert call(E=3, H=260, W=346, bins=5) == binding.EVIS_ERR_TOO_LARGE
    assert call(E=65535, H=32767, W=32767, bins=2 ** 31 - 1) == binding.EVIS_ERR_TOO_LARGE
    assert call(E=1, H=1024, W=1025, bins=1) == binding.EVIS_ERR_TOO_LARGE            # one column beyond the limit
    assert err.value == 0
    assert b"evis_voxelize_static" in L.evis_strerror(binding.EVIS_ERR_TOO_LARGE)
    src = open(binding.LIB_PATH.replace("libevis.so", "../include/evis.h")).read()
    assert f"#define EVIS_VOXELIZE_STATIC_MAX_CELLS (1u << {binding.VOXELIZE_STATIC_MAX_CELLS.bit_length() - 1})" in src


def _existing_path(spec, bins, window, margin=0):
    """The context's own grid (evis_set_voxels) over one window, raw and normalised, plus the window's events."""
    sc = scenes.make_scene(spec)
    ev = binding.Evis(spec.num_envs, spec.height, spec.width, spec.substeps, spec.c_pos, spec.c_neg, spec.log_eps,
                      spec.keyframe_dt, max_motion_px=spec.max_motion_px(), event_capacity=1 << 23)
    if margin:
        ev.set_margin(margin)
    ev.set_voxels(bins, window_steps=window, keep_events=True)
    events = []
    try:
        for k in range(window + 1):
            kf = scenes.render_keyframe(sc, k, device="cuda")
            ev.step(kf["rad"], kf["mv_bwd"], kf["depth"], mv_fwd=kf["mv_fwd"], sync=True)
            if k:
                events.append(ev.read_events().copy())
        raw, n = ev.read_voxels()
        assert n == window
        norm, _ = ev.read_voxels(normalize=True)
    finally:
        ev.destroy()
    return np.concatenate(events), raw, norm


@pytest.mark.gpu
def test_static_voxel_grid_equals_the_contexts_grid_on_two_calls_in_a_row():
    dev = torch.device("cuda", 0)
    # call 1: three environments, a window of three intervals, five bins (every event lands in two bins)
    spec1 = scenes.small(scenes.config(4), num_envs=3, height=97, width=131, num_keyframes=4)
    e1, raw1, norm1 = _existing_path(spec1, bins=5, window=3)
    # call 2: another scene and shape, fewer cells, over-render margin (the grid has the cropped frame's shape)
    spec2 = scenes.small(scenes.config(2), num_envs=2, height=70, width=90, num_keyframes=3)
    e2, raw2, norm2 = _existing_path(spec2, bins=2, window=2, margin=4)
    assert len(e1) > 1000 and len(e2) > 1000 and set(np.unique(e1["kf"])) == {0, 1, 2}

    def to_device(e):
        return torch.from_numpy(e.view(np.uint8).reshape(-1, 16).copy()).to(dev)

    d1, d2 = to_device(e1), to_device(e2)
    # the caller brings the outputs; poisoned so that an unwritten cell shows
    g1 = torch.full(raw1.shape, float("nan"), dtype=torch.float32, device=dev)
    g2 = torch.full(raw2.shape, float("nan"), dtype=torch.float32, device=dev)
    g2n = torch.full(raw2.shape, float("nan"), dtype=torch.float32, device=dev)
    g1n = torch.full(raw1.shape, float("nan"), dtype=torch.float32, device=dev)
    torch.cuda.synchronize(dev)
    # back to back on one stream, nothing waited for in between: the calls are ordered on the GPU and share the array
    binding.voxelize_static(d1, g1, window_steps=3, keyframe_dt=spec1.keyframe_dt)
    binding.voxelize_static(d2, g2, window_steps=2, keyframe_dt=spec2.keyframe_dt)
    binding.voxelize_static(d2, g2n, window_steps=2, keyframe_dt=spec2.keyframe_dt, normalize=True)
    binding.voxelize_static(d1, g1n, window_steps=3, keyframe_dt=spec1.keyframe_dt, normalize=True)
    torch.cuda.synchronize(dev)
    # tolerance: none needed -- the same arithmetic on integer sums; np.array_equal is inside every tolerance of the voxel tests
    assert np.array_equal(g1.cpu().numpy(), raw1)
    assert np.array_equal(g2.cpu().numpy(), raw2)
    assert np.array_equal(g2n.cpu().numpy(), norm2)
    assert np.array_equal(g1n.cpu().numpy(), norm1)
    assert abs(float(raw1.astype(np.float64).sum()) - len(e1)) < 0.5 and float(norm1.max()) == 1.0       # the comparison is not vacuous
    # once its kernels are loaded (the calls above), a call takes no device memory at all
    free_mid = torch.cuda.mem_get_info(dev)[0]
    binding.voxelize_static(d2, g2, window_steps=2, keyframe_dt=spec2.keyframe_dt)
    torch.cuda.synchronize(dev)
    assert torch.cuda.mem_get_info(dev)[0] == free_mid
    assert np.array_equal(g2.cpu().numpy(), raw2)

    # a window that does not start at interval 0, and events outside it / outside the frame / of an env beyond E: ignored
    sel = e1[e1["kf"] >= 1].copy()
    junk = sel[:64].copy()
    junk["kf"][:16] = 7; junk["x"][16:32] = 500; junk["y"][32:48] = 400; junk["env"][48:] = 9
    sc = scenes.make_scene(spec1)
    ev = binding.Evis(spec1.num_envs, spec1.height, spec1.width, spec1.substeps, spec1.c_pos, spec1.c_neg, spec1.log_eps,
                      spec1.keyframe_dt, max_motion_px=spec1.max_motion_px(), event_capacity=1 << 23)
    try:
        for k in range(4):
            if k == 2:
                ev.set_voxels(4, window_steps=2)       # the window opens with interval 1
            kf = scenes.render_keyframe(sc, k, device="cuda")
            ev.step(kf["rad"], kf["mv_bwd"], kf["depth"], mv_fwd=kf["mv_fwd"], sync=True)
        want, n = ev.read_voxels()
        assert n == 2
    finally:
        ev.destroy()
    g = torch.full(want.shape, float("nan"), dtype=torch.float32, device=dev)
    binding.voxelize_static(to_device(np.concatenate([junk, sel])), g, window_steps=2, keyframe_dt=spec1.keyframe_dt, first_kf=1)
    torch.cuda.synchronize(dev)
    assert np.array_equal(g.cpu().numpy(), want)

    # no events: a grid of zeros; too large: refused, the output untouched
    binding.voxelize_static(d1[:0], g, window_steps=2, keyframe_dt=spec1.keyframe_dt)
    torch.cuda.synchronize(dev)
    assert float(g.abs().max()) == 0.0
    big = torch.full((3, 2, 5, 260, 346), 3.0, dtype=torch.float32, device=dev)
    with pytest.raises(binding.EvisError) as ei:
        binding.voxelize_static(d1, big, window_steps=3, keyframe_dt=spec1.keyframe_dt)
    assert ei.value.status == binding.EVIS_ERR_TOO_LARGE
    torch.cuda.synchronize(dev)
    assert float(big.min()) == 3.0 and float(big.max()) == 3.0
