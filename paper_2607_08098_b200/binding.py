"""Thin ctypes binding of the C ABI in include/evis.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libevis.so.  There is NO CPU fallback: if the
library is missing or does not load, importing a symbol from it raises.  PyTorch is used for device
memory and streams (tensors in, tensors out).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Tuple

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libevis.so")

EVIS_OK = 0
EVIS_ERR_INVALID_ARG, EVIS_ERR_CUDA, EVIS_ERR_OOM = -1, -2, -3
EVIS_ERR_OVERFLOW, EVIS_ERR_MOTION_BOUND, EVIS_ERR_BAD_STATE = -4, -5, -6
EVIS_ERR_TOO_LARGE = -7
VOXELIZE_STATIC_MAX_CELLS = 1 << 21      # EVIS_VOXELIZE_STATIC_MAX_CELLS of include/evis.h
PATH_AUTO, PATH_GLOBAL = 0, 1
COMPOSITE_B_PRIMARY, COMPOSITE_BLEND, COMPOSITE_WEIGHTED = 0, 1, 2

EVENT_DTYPE = np.dtype([("x", "<u2"), ("y", "<u2"), ("env", "<u2"), ("p", "i1"), ("substep", "u1"),
                        ("t_off", "<f4"), ("kf", "<u4")])
assert EVENT_DTYPE.itemsize == 16


class evis_config(C.Structure):
    _fields_ = [("num_envs", C.c_int32), ("height", C.c_int32), ("width", C.c_int32), ("substeps", C.c_int32),
                ("c_pos", C.c_float), ("c_neg", C.c_float), ("log_eps", C.c_float), ("keyframe_dt", C.c_float),
                ("max_motion_px", C.c_float), ("composite_mode", C.c_int32), ("path", C.c_int32),
                ("device", C.c_int32), ("event_capacity", C.c_uint64), ("debug_capture", C.c_int32),
                ("reserved", C.c_int32)]


class evis_info(C.Structure):
    _fields_ = [("path", C.c_int32), ("tile_w", C.c_int32), ("tile_h", C.c_int32), ("halo", C.c_int32),
                ("steps", C.c_uint64), ("last_events", C.c_uint64), ("last_holes", C.c_uint64),
                ("kernel_launches", C.c_uint64), ("last_overflow", C.c_int32),
                ("last_motion_violation", C.c_int32), ("device_bytes", C.c_uint64), ("total_events", C.c_uint64),
                ("overflow_steps", C.c_uint64)]


NUM_STAGES = 8
STAGE_NAMES = ["prep", "clear", "splat", "resolve", "order", "s5", "splat+resolve", "s7"]


class evis_profile(C.Structure):
    _fields_ = [("steps", C.c_uint64), ("launches", C.c_uint64 * NUM_STAGES), ("ms", C.c_double * NUM_STAGES)]


# every symbol include/evis.h declares (tests/test_abi.py checks the list against the header)
SYMBOLS = ["evis_create", "evis_step", "evis_step_host", "evis_read_events", "evis_events_device",
           "evis_get_info", "evis_profile_enable", "evis_profile_read", "evis_get_state", "evis_set_state", "evis_debug_read", "evis_destroy",
           "evis_strerror", "evis_last_cuda_error", "evis_version", "evis_set_thresholds", "evis_set_refractory", "evis_set_margin", "evis_set_channel", "evis_set_noise", "evis_wait_events", "evis_refractory_state", "evis_read_events_begin", "evis_read_events_end",
           "evis_set_interval_index", "evis_set_voxels", "evis_read_voxels", "evis_read_voxels_begin", "evis_read_voxels_end", "evis_set_defocus", "evis_set_time_sorted", "evis_set_compact_events", "evis_read_events8", "evis_read_events8_begin",
           "evis_voxelize_static", "evis_set_env_offset",
           "evis_read_events_enqueue", "evis_read_events_finish"]

_lib = None


def load() -> C.CDLL:
    """Load libevis.so.  Raises if it has not been built (python -m paper_2607_08098_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2607_08098_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, u64p = C.c_void_p, C.POINTER(C.c_uint64)
    L.evis_create.argtypes = [C.POINTER(evis_config), C.POINTER(vp)]
    L.evis_step.argtypes = [vp, vp, vp, vp, vp, vp, u64p]
    L.evis_step_host.argtypes = [vp, vp, vp, vp, vp, u64p]
    L.evis_read_events.argtypes = [vp, vp, C.c_int, C.c_uint64, u64p]
    L.evis_events_device.argtypes = [vp, C.POINTER(vp), u64p]
    L.evis_get_info.argtypes = [vp, C.POINTER(evis_info)]
    L.evis_profile_enable.argtypes = [vp, C.c_int]
    L.evis_profile_read.argtypes = [vp, C.POINTER(evis_profile)]
    L.evis_get_state.argtypes = [vp, vp, vp]
    L.evis_set_state.argtypes = [vp, vp, vp]
    L.evis_debug_read.argtypes = [vp, vp, vp, vp]
    L.evis_destroy.argtypes = [vp]
    L.evis_strerror.argtypes = [C.c_int]
    L.evis_strerror.restype = C.c_char_p
    L.evis_set_thresholds.argtypes = [vp, vp, vp, C.c_int]
    L.evis_set_refractory.argtypes = [vp, C.c_float]
    L.evis_set_margin.argtypes = [vp, C.c_int]
    L.evis_set_channel.argtypes = [vp, C.c_int]
    L.evis_set_interval_index.argtypes = [vp, C.c_uint32]
    L.evis_set_env_offset.argtypes = [vp, C.c_uint32]
    L.evis_wait_events.argtypes = [vp, vp]
    L.evis_read_events_begin.argtypes = [vp, vp, C.c_uint64, u64p]
    L.evis_read_events_end.argtypes = [vp]
    L.evis_read_events_enqueue.argtypes = [vp, vp, C.c_uint64, C.c_int]
    L.evis_read_events_finish.argtypes = [vp, u64p]
    L.evis_refractory_state.argtypes = [vp, vp, vp]
    L.evis_set_noise.argtypes = [vp, C.POINTER(evis_noise), vp, C.c_int]
    L.evis_set_voxels.argtypes = [vp, C.POINTER(evis_voxel_config)]
    L.evis_read_voxels.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_uint32)]
    L.evis_read_voxels_begin.argtypes = [vp, vp, C.c_int, C.c_int]
    L.evis_read_voxels_end.argtypes = [vp]
    L.evis_set_defocus.argtypes = [vp, C.c_float]
    L.evis_set_time_sorted.argtypes = [vp, C.c_int]
    L.evis_set_compact_events.argtypes = [vp, C.c_int]
    L.evis_read_events8.argtypes = [vp, vp, C.c_int, C.c_uint64, u64p]
    L.evis_read_events8_begin.argtypes = [vp, vp, C.c_uint64, u64p]
    L.evis_voxelize_static.argtypes = [vp, C.c_uint64, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_float,
                                       C.c_uint32, C.c_int, vp, vp, C.POINTER(C.c_int)]
    L.evis_last_cuda_error.argtypes = [vp]
    L.evis_version.restype = C.c_char_p
    for name in SYMBOLS:
        getattr(L, name)              # raises AttributeError if the library lacks a declared symbol
    _lib = L
    return L


class evis_voxel_config(C.Structure):
    _fields_ = [("bins", C.c_int32), ("window_steps", C.c_int32), ("keep_events", C.c_int32), ("reserved", C.c_int32)]


class evis_noise(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("r_leak", C.c_float), ("r_shot", C.c_float), ("r_hot", C.c_float),
                ("i_white", C.c_float)]


class EvisError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {load().evis_strerror(status).decode()} ({status})")


def _check(status: int, where: str, allow=()):
    if status != EVIS_OK and status not in allow:
        raise EvisError(status, where)
    return status


def _dev_ptr(t: Optional[torch.Tensor], shape: Tuple[int, ...], name: str) -> Optional[int]:
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
        raise ValueError(f"{name}: need a contiguous float32 CUDA tensor of shape {shape}")
    return t.data_ptr()


def _host_ptr(t, shape, name) -> Optional[int]:
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        if not (t.dtype == np.float32 and t.flags.c_contiguous and tuple(t.shape) == tuple(shape)):
            raise ValueError(f"{name}: need a C-contiguous float32 array of shape {shape}")
        return t.ctypes.data
    if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: need a contiguous float32 CPU tensor of shape {shape}")
    return t.data_ptr()


class Evis:
    """One context of the library (evis_create .. evis_destroy); method names follow the ABI."""

    def __init__(self, num_envs: int, height: int, width: int, substeps: int, c_pos: float, c_neg: float,
                 log_eps: float, keyframe_dt: float, max_motion_px: float = 0.0, composite_mode: int = 0,
                 path: int = PATH_AUTO, device: int = 0, event_capacity: int = 1 << 22,
                 debug_capture: bool = False):
        self._lib = load()
        self.cfg = evis_config(num_envs, height, width, substeps, c_pos, c_neg, log_eps, keyframe_dt,
                               max_motion_px, composite_mode, path, device, event_capacity,
                               int(debug_capture), 0)
        self._ctx = C.c_void_p()
        _check(self._lib.evis_create(C.byref(self.cfg), C.byref(self._ctx)), "evis_create")
        self.E, self.H, self.W, self.S = num_envs, height, width, substeps
        self.device = device

    # -- evis_step ---------------------------------------------------------------------------------
    def step(self, rad: torch.Tensor, mv_bwd: torch.Tensor, depth: torch.Tensor,
             mv_fwd: Optional[torch.Tensor] = None, sync: bool = False, stream: Optional[torch.cuda.Stream] = None,
             allow=()) -> Optional[int]:
        """Enqueue one keyframe on ``stream`` (default: torch's current stream).  With ``sync`` the call
        waits and returns the true event count of the step."""
        E, H, W = self.E, self.H, self.W
        st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
        n = C.c_uint64(0)
        rc = self._lib.evis_step(self._ctx, _dev_ptr(rad, (E, H, W, 3), "rad"), _dev_ptr(mv_bwd, (E, H, W, 2), "mv_bwd"),
                                 _dev_ptr(mv_fwd, (E, H, W, 2), "mv_fwd"), _dev_ptr(depth, (E, H, W), "depth"),
                                 C.c_void_p(st), C.byref(n) if sync else None)
        _check(rc, "evis_step", allow)
        return int(n.value) if sync else None

    def set_thresholds(self, theta_on: Optional[torch.Tensor], theta_off: Optional[torch.Tensor]) -> None:
        """evis_set_thresholds (Eq. 8): per-pixel ON / OFF threshold maps [E,H,W] float32, CUDA tensors on this
        context's device; both None = back to the scalar thresholds.  The library copies them."""
        if theta_on is None and theta_off is None:
            _check(self._lib.evis_set_thresholds(self._ctx, None, None, 1), "evis_set_thresholds")
            return
        E, H, W = self.E, self.H, self.W
        p_on, p_off = _dev_ptr(theta_on, (E, H, W), "theta_on"), _dev_ptr(theta_off, (E, H, W), "theta_off")
        torch.cuda.synchronize(self.device)                 # the library copies on its own stream
        _check(self._lib.evis_set_thresholds(self._ctx, p_on, p_off, 1), "evis_set_thresholds")

    def set_noise(self, seed: int = 0, r_leak: float = 0.0, r_shot: float = 0.0, r_hot: float = 0.0,
                  i_white: float = 1.0, hot: Optional[torch.Tensor] = None, off: bool = False) -> None:
        """evis_set_noise (Eq. 9-10 and hot pixels): rates in Hz; ``hot`` = uint8 CUDA tensor [E,H,W] or None;
        ``off=True`` switches the noise events off."""
        if off:
            _check(self._lib.evis_set_noise(self._ctx, None, None, 1), "evis_set_noise")
            return
        cfg = evis_noise(int(seed), float(r_leak), float(r_shot), float(r_hot), float(i_white))
        hp = None
        if hot is not None:
            if not (hot.is_cuda and hot.dtype == torch.uint8 and hot.is_contiguous() and tuple(hot.shape) == (self.E, self.H, self.W)):
                raise ValueError("hot: need a contiguous uint8 CUDA tensor of shape (E, H, W)")
            torch.cuda.synchronize(self.device)
            hp = hot.data_ptr()
        _check(self._lib.evis_set_noise(self._ctx, C.byref(cfg), hp, 1), "evis_set_noise")

    def set_voxels(self, bins: Optional[int], window_steps: int = 1, keep_events: bool = True) -> None:
        """evis_set_voxels: per-polarity voxel grid [E, 2, bins, H', W'] over windows of `window_steps` intervals
        (PAPER.md:331); bins = None switches it off."""
        if bins is None:
            _check(self._lib.evis_set_voxels(self._ctx, None), "evis_set_voxels")
            self._vox = None
            return
        cfg = evis_voxel_config(int(bins), int(window_steps), int(bool(keep_events)), 0)
        _check(self._lib.evis_set_voxels(self._ctx, C.byref(cfg)), "evis_set_voxels")
        self._vox = int(bins)

    def voxel_shape(self) -> Tuple[int, int, int, int, int]:
        m = getattr(self, "_margin", 0)
        return (self.E, 2, self._vox, self.H - 2 * m, self.W - 2 * m)

    def read_voxels(self, normalize: bool = False, restart: bool = False) -> Tuple[np.ndarray, int]:
        """evis_read_voxels to a new host array; returns (grid float32, intervals accumulated in the window)."""
        out = np.empty(self.voxel_shape(), np.float32)
        n = C.c_uint32(0)
        _check(self._lib.evis_read_voxels(self._ctx, out.ctypes.data, 0, int(normalize), int(restart), C.byref(n)),
               "evis_read_voxels")
        return out, int(n.value)

    def read_voxels_begin(self, host_buf: np.ndarray, normalize: bool = False, restart: bool = False) -> None:
        assert host_buf.dtype == np.float32 and host_buf.flags.c_contiguous and host_buf.size == int(np.prod(self.voxel_shape()))
        _check(self._lib.evis_read_voxels_begin(self._ctx, host_buf.ctypes.data, int(normalize), int(restart)),
               "evis_read_voxels_begin")

    def read_voxels_end(self) -> None:
        _check(self._lib.evis_read_voxels_end(self._ctx), "evis_read_voxels_end")

    def set_time_sorted(self, on: bool = True) -> None:
        """evis_set_time_sorted: the stored stream of later steps is ordered by (env, t_off), stable."""
        _check(self._lib.evis_set_time_sorted(self._ctx, int(bool(on))), "evis_set_time_sorted")

    def set_compact_events(self, on: bool = True) -> None:
        """evis_set_compact_events: the stored stream holds 8-byte events (read them with read_events8)."""
        _check(self._lib.evis_set_compact_events(self._ctx, int(bool(on))), "evis_set_compact_events")

    def read_events8(self, max_events: Optional[int] = None, allow=()) -> np.ndarray:
        """evis_read_events8 to a new host array of uint64 (decode with ``decode_events8``)."""
        n = min(int(self.info().last_events), int(self.cfg.event_capacity))
        if max_events is not None:
            n = min(n, int(max_events))
        out = np.empty(n, np.uint64)
        got = C.c_uint64(0)
        _check(self._lib.evis_read_events8(self._ctx, out.ctypes.data if n else None, 0, n, C.byref(got)), "evis_read_events8", allow)
        return out[:got.value]

    def read_events8_begin(self, host_buf: np.ndarray) -> int:
        assert host_buf.dtype == np.uint64 and host_buf.flags.c_contiguous
        got = C.c_uint64(0)
        _check(self._lib.evis_read_events8_begin(self._ctx, host_buf.ctypes.data, host_buf.size, C.byref(got)), "evis_read_events8_begin")
        return int(got.value)

    def set_defocus(self, sigma: float) -> None:
        """evis_set_defocus: Gaussian blur of the warped linear frame before the event model."""
        _check(self._lib.evis_set_defocus(self._ctx, float(sigma)), "evis_set_defocus")

    def set_channel(self, channel: int) -> None:
        """evis_set_channel (colour events): 0 / 1 / 2 = log of R / G / B, -1 = Rec.709 luminance."""
        _check(self._lib.evis_set_channel(self._ctx, int(channel)), "evis_set_channel")

    def set_interval_index(self, next_kf: int) -> None:
        """evis_set_interval_index: the index the next closed interval gets (checkpoint / resume)."""
        _check(self._lib.evis_set_interval_index(self._ctx, int(next_kf)), "evis_set_interval_index")

    def set_env_offset(self, first_env: int) -> None:
        """evis_set_env_offset: this context holds envs [first_env, first_env + E) of a larger batch (keys the noise events)."""
        _check(self._lib.evis_set_env_offset(self._ctx, int(first_env)), "evis_set_env_offset")

    def set_margin(self, margin: int) -> None:
        """evis_set_margin: the frames carry `margin` over-rendered pixels per side, cropped after the warp."""
        _check(self._lib.evis_set_margin(self._ctx, int(margin)), "evis_set_margin")
        self._margin = int(margin)

    def set_refractory(self, tau_r: float) -> None:
        """evis_set_refractory: refractory period in seconds, 0 = off; resets the per-pixel state."""
        _check(self._lib.evis_set_refractory(self._ctx, float(tau_r)), "evis_set_refractory")

    def wait_events(self, stream: Optional[torch.cuda.Stream] = None) -> None:
        """evis_wait_events: make ``stream`` (default: torch's current stream) wait for the last step's ordered stream."""
        st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
        _check(self._lib.evis_wait_events(self._ctx, C.c_void_p(st)), "evis_wait_events")

    def step_host(self, rad, mv_bwd, depth, mv_fwd=None, allow=(), sync: bool = True) -> Optional[int]:
        """evis_step_host: HOST buffers (numpy or CPU tensors).  sync: wait for the step and return its event count;
        else return once the upload is done (the step keeps running and overlaps the next upload)."""
        E, H, W = self.E, self.H, self.W
        n = C.c_uint64(0)
        rc = self._lib.evis_step_host(self._ctx, _host_ptr(rad, (E, H, W, 3), "rad"),
                                      _host_ptr(mv_bwd, (E, H, W, 2), "mv_bwd"),
                                      _host_ptr(mv_fwd, (E, H, W, 2), "mv_fwd"),
                                      _host_ptr(depth, (E, H, W), "depth"), C.byref(n) if sync else None)
        _check(rc, "evis_step_host", allow)
        return int(n.value) if sync else None

    # -- evis_read_events --------------------------------------------------------------------------
    def read_events(self, max_events: Optional[int] = None, allow=()) -> np.ndarray:
        """Events of the last step in the library's deterministic order (host structured array).  After a step that
        overflowed the call raises EVIS_ERR_OVERFLOW unless ``allow`` lists it; the valid prefix is returned then."""
        info = self.info()
        n = min(info.last_events, self.cfg.event_capacity)
        if max_events is not None:
            n = min(n, max_events)
        out = np.empty(n, dtype=EVENT_DTYPE)
        got = C.c_uint64(0)
        _check(self._lib.evis_read_events(self._ctx, out.ctypes.data if n else None, 0, n, C.byref(got)),
               "evis_read_events", allow)
        return out[:got.value]

    def read_events_into(self, host_buf: np.ndarray) -> int:
        """evis_read_events into a preallocated (e.g. pinned) host buffer of EVENT_DTYPE."""
        got = C.c_uint64(0)
        _check(self._lib.evis_read_events(self._ctx, host_buf.ctypes.data, 0, host_buf.shape[0], C.byref(got)),
               "evis_read_events")
        return int(got.value)

    def read_events_begin(self, host_buf: np.ndarray) -> int:
        """evis_read_events_begin: start copying the last step's events into a (pinned) host buffer; returns their number."""
        got = C.c_uint64(0)
        _check(self._lib.evis_read_events_begin(self._ctx, host_buf.ctypes.data, host_buf.shape[0], C.byref(got)),
               "evis_read_events_begin")
        return int(got.value)

    def read_events_enqueue(self, pinned_buf: np.ndarray, previous_step: bool = False) -> None:
        """evis_read_events_enqueue: start copying the stored stream of the last step -- or, with ``previous_step``, of the step
        before it, waiting only for that one (the pipelined loop) -- into a PINNED host array (EVENT_DTYPE, or uint64 with
        compact events); ``read_events_finish`` waits for the copy and returns how many events arrived."""
        assert pinned_buf.flags.c_contiguous and pinned_buf.dtype.itemsize in (8, 16)
        _check(self._lib.evis_read_events_enqueue(self._ctx, pinned_buf.ctypes.data, pinned_buf.shape[0], int(bool(previous_step))),
               "evis_read_events_enqueue")

    def read_events_finish(self, allow=()) -> int:
        got = C.c_uint64(0)
        _check(self._lib.evis_read_events_finish(self._ctx, C.byref(got)), "evis_read_events_finish", allow)
        return int(got.value)

    def read_events_end(self) -> None:
        _check(self._lib.evis_read_events_end(self._ctx), "evis_read_events_end")

    def events_device(self) -> Tuple[int, int]:
        """(device pointer, stored count) of the ordered stream of the last step; no copy."""
        p, n = C.c_void_p(), C.c_uint64(0)
        _check(self._lib.evis_events_device(self._ctx, C.byref(p), C.byref(n)), "evis_events_device")
        return int(p.value or 0), int(n.value)

    # -- info / state / debug ----------------------------------------------------------------------
    def info(self) -> evis_info:
        i = evis_info()
        _check(self._lib.evis_get_info(self._ctx, C.byref(i)), "evis_get_info")
        return i

    def profile_enable(self, on: bool = True) -> None:
        _check(self._lib.evis_profile_enable(self._ctx, int(on)), "evis_profile_enable")

    def profile_read(self) -> dict:
        """{'steps': n, 'ms': {stage: device ms summed}, 'launches': {stage: count}} since the last read."""
        p = evis_profile()
        _check(self._lib.evis_profile_read(self._ctx, C.byref(p)), "evis_profile_read")
        return {"steps": int(p.steps),
                "ms": {STAGE_NAMES[i]: float(p.ms[i]) for i in range(NUM_STAGES) if p.launches[i]},
                "launches": {STAGE_NAMES[i]: int(p.launches[i]) for i in range(NUM_STAGES) if p.launches[i]}}

    def get_state(self) -> Tuple[np.ndarray, np.ndarray]:
        shp = (self.E, self.H, self.W)
        lref, lprev = np.empty(shp, np.float32), np.empty(shp, np.float32)
        _check(self._lib.evis_get_state(self._ctx, lref.ctypes.data, lprev.ctypes.data), "evis_get_state")
        return lref, lprev

    def get_t_last(self) -> np.ndarray:
        """evis_refractory_state (get): stamps of the last emitted events, relative to the next interval's start."""
        out = np.empty((self.E, self.H, self.W), np.float32)
        _check(self._lib.evis_refractory_state(self._ctx, out.ctypes.data, None), "evis_refractory_state")
        return out

    def set_t_last(self, t_last: np.ndarray) -> None:
        _check(self._lib.evis_refractory_state(self._ctx, None, _host_ptr(t_last, (self.E, self.H, self.W), "t_last")),
               "evis_refractory_state")

    def set_state(self, l_ref: Optional[np.ndarray], l_prev: Optional[np.ndarray]) -> None:
        shp = (self.E, self.H, self.W)
        _check(self._lib.evis_set_state(self._ctx, _host_ptr(l_ref, shp, "l_ref"), _host_ptr(l_prev, shp, "l_prev")),
               "evis_set_state")

    def debug_read(self):
        """(win [S,E,H,W] u32, dir [S,E,H,W] u8, l_hat [S,E,H,W] f32) of the last step."""
        shp = (self.S, self.E, self.H, self.W)
        win, d, lh = np.empty(shp, np.uint32), np.empty(shp, np.uint8), np.empty(shp, np.float32)
        _check(self._lib.evis_debug_read(self._ctx, win.ctypes.data, d.ctypes.data, lh.ctypes.data), "evis_debug_read")
        return win, d, lh

    def destroy(self) -> None:
        if self._ctx:
            self._lib.evis_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def voxelize_static(events: torch.Tensor, grid: torch.Tensor, window_steps: int, keyframe_dt: float, first_kf: int = 0,
                    normalize: bool = False, stream: Optional[torch.cuda.Stream] = None) -> None:
    """evis_voxelize_static: the voxel grid of finished events WITHOUT any device allocation -- for code that runs where
    cudaMalloc is off limits (a rollout loop whose memory was shared out among the simulator's, the renderer's and the
    learner's pools beforehand, and where an allocation would also stall every stream of the GPU) and so cannot use
    ``Evis.set_voxels``.  The caller owns both tensors, and this wrapper creates none: ``events`` is a contiguous CUDA
    tensor of 16-byte evis_event records (uint8 [n, 16] or int32 [n, 4]; n may be 0), ``grid`` a contiguous float32 CUDA
    tensor [E, 2, bins, H, W] on the same device, overwritten.  The accumulator in between is a fixed 16 MiB array inside
    the library, shared by all calls on a GPU: E * 2 * bins * H * W may not exceed ``VOXELIZE_STATIC_MAX_CELLS``
    (EvisError with EVIS_ERR_TOO_LARGE otherwise), and calls whose GPU work can overlap (unordered streams) must be
    serialised by the caller.  Only enqueues on ``stream`` (default: torch's current stream of that device).  The first
    call on a device also does the library's one-time address look-up: make it before any stream capture."""
    if not (events.is_cuda and events.is_contiguous() and events.dim() == 2 and
            events.shape[1] * events.element_size() == 16 and events.data_ptr() % 16 == 0):
        raise ValueError("events: need a contiguous, 16-byte aligned CUDA tensor of 16-byte records, shape [n, 16 / itemsize]")
    if not (grid.is_cuda and grid.dtype == torch.float32 and grid.is_contiguous() and grid.dim() == 5 and grid.shape[1] == 2
            and grid.device == events.device):
        raise ValueError("grid: need a contiguous float32 CUDA tensor [E, 2, bins, H, W] on the events' device")
    E, _, bins, H, W = (int(v) for v in grid.shape)
    err = C.c_int(0)
    with torch.cuda.device(grid.device):            # the library uses the current device's copy of its array
        st = (stream or torch.cuda.current_stream(grid.device)).cuda_stream
        rc = load().evis_voxelize_static(events.data_ptr() if events.shape[0] else None, int(events.shape[0]), E, H, W, bins,
                                         int(window_steps), float(keyframe_dt), int(first_kf), int(bool(normalize)),
                                         grid.data_ptr(), C.c_void_p(st), C.byref(err))
    _check(rc, f"evis_voxelize_static (cudaError {err.value})" if err.value else "evis_voxelize_static")


def decode_events8(ev8: np.ndarray, keyframe_dt: float, substeps: int, kf: int = 0) -> np.ndarray:
    """8-byte events (include/evis.h, evis_event8) -> the 16-byte record layout (EVENT_DTYPE); t_off is the centre of the
    stamp's 2^-15 cell of its substep."""
    ev8 = np.asarray(ev8, np.uint64)
    out = np.zeros(len(ev8), EVENT_DTYPE)
    out["x"] = (ev8 & np.uint64(0xFFF)).astype(np.uint16)
    out["y"] = ((ev8 >> np.uint64(12)) & np.uint64(0xFFF)).astype(np.uint16)
    out["env"] = ((ev8 >> np.uint64(24)) & np.uint64(0xFFFF)).astype(np.uint16)
    sub = ((ev8 >> np.uint64(40)) & np.uint64(0xFF)).astype(np.int64)
    out["substep"] = sub.astype(np.uint8)
    frac = ((ev8 >> np.uint64(48)) & np.uint64(0x7FFF)).astype(np.float64)
    out["p"] = np.where((ev8 >> np.uint64(63)) != 0, 1, -1).astype(np.int8)
    out["t_off"] = ((sub - 1) + (frac + 0.5) / 32768.0) * (keyframe_dt / substeps)
    out["kf"] = kf
    return out
