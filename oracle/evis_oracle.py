"""ctypes front end of the C oracle (oracle/evis_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares nothing with the CUDA path; it mirrors the library's call shape
(first keyframe initialises, every later keyframe closes one interval A -> B) so
that the parity tests can feed both sides the same keyframes.
"""
from __future__ import annotations

import ctypes as C
from typing import Dict, Optional

import numpy as np

from . import build as _build

class Noise(C.Structure):
    """evo_noise (oracle/evis_oracle.c): parameters of the noise events, Eq. 9-10 and hot pixels [R29]."""
    _fields_ = [("seed", C.c_uint64), ("r_leak", C.c_float), ("r_shot", C.c_float), ("r_hot", C.c_float),
                ("i_white", C.c_float), ("eps", C.c_float), ("hot", C.c_void_p)]


EVENT_DTYPE = np.dtype([("env", "<i4"), ("x", "<i4"), ("y", "<i4"), ("p", "<i4"), ("substep", "<i4"),
                        ("k", "<i4"), ("kf", "<i4"), ("pad", "<i4"), ("t_off", "<f8")])
NONE = 0xFFFFFFFF

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        fp, u64p, u32p, u8p = (C.POINTER(C.c_float), C.POINTER(C.c_uint64), C.POINTER(C.c_uint32),
                               C.POINTER(C.c_uint8))
        L.evo_log_luminance.argtypes = [fp, C.c_int64, C.c_float, fp]
        L.evo_log_luminance.restype = None
        L.evo_log_channel.argtypes = [fp, C.c_int64, C.c_float, C.c_int, fp]
        L.evo_log_channel.restype = None
        L.evo_splat.argtypes = [C.c_int] * 5 + [fp, fp, fp, u64p]
        L.evo_splat.restype = None
        L.evo_composite.argtypes = [C.c_int] * 5 + [u64p, u64p, fp, fp, fp, fp, u8p, u32p]
        L.evo_composite.restype = None
        L.evo_event_frame.argtypes = [C.c_int] * 6 + [C.c_float] * 3 + [fp, fp] + [C.c_float, fp] + [C.c_void_p] + [fp, fp, fp, C.c_void_p,
                                                                        C.c_int64, C.c_int64, fp]
        L.evo_event_frame.restype = C.c_int64
        L.evo_interval.argtypes = ([C.c_int] * 7 + [C.c_float] * 3 + [fp, fp] + [C.c_float, fp] + [C.c_void_p] + [fp] * 8 + [u64p, u64p, fp]
                                   + [C.c_void_p, C.c_int64, C.c_int64]
                                   + [u32p, u32p, u8p, u32p, fp, fp, C.POINTER(C.c_int64)]
                                   + [C.c_int, fp, fp, fp, fp, C.c_float, fp, fp]
                                   + [C.POINTER(C.c_int64), C.POINTER(C.c_int64)])
        L.evo_interval.restype = C.c_int64
        L.evo_wsplat.argtypes = [C.c_int] * 5 + [fp, fp, fp, fp, u64p, C.POINTER(C.c_int64)]
        L.evo_wsplat.restype = None
        L.evo_linear_luminance.argtypes = [fp, C.c_int64, C.c_int, fp]
        L.evo_linear_luminance.restype = None
        L.evo_gauss_taps.argtypes = [C.c_float, fp, C.c_int]
        L.evo_gauss_taps.restype = C.c_int
        L.evo_blur.argtypes = [C.c_int, C.c_int, C.c_int, fp, fp, fp, fp]
        L.evo_blur.restype = None
        L.evo_exp32.argtypes = [C.c_float]
        L.evo_exp32.restype = C.c_float
        L.evo_noise_key.argtypes = [C.c_uint64, C.c_int, C.c_int, C.c_int64]
        L.evo_noise_key.restype = C.c_uint64
        L.evo_noise_hash.argtypes = [C.c_uint64, C.c_int, C.c_int]
        L.evo_noise_hash.restype = C.c_uint64
        _lib = L
    return _lib


def _f(a):
    assert a.dtype == np.float32 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def log_luminance(rad: np.ndarray, eps: float, channel: Optional[int] = None) -> np.ndarray:
    """Eq. 3 + log.  rad [...,3] float32 -> L [...] float32.
    channel = 0 / 1 / 2: colour events: the log of that channel instead of the luminance."""
    rad = np.ascontiguousarray(rad, dtype=np.float32)
    out = np.empty(rad.shape[:-1], dtype=np.float32)
    if channel is None:
        lib().evo_log_luminance(_f(rad), out.size, float(eps), _f(out))
    else:
        assert channel in (0, 1, 2)
        lib().evo_log_channel(_f(rad), out.size, float(eps), int(channel), _f(out))
    return out


def linear_luminance(rad: np.ndarray, channel: Optional[int] = None) -> np.ndarray:
    """Linear intensity of Eq. 3 (or of one channel), clamped at 0, float32 [R31].  rad [...,3] -> I [...]."""
    rad = np.ascontiguousarray(rad, dtype=np.float32)
    out = np.empty(rad.shape[:-1], dtype=np.float32)
    lib().evo_linear_luminance(_f(rad), out.size, -1 if channel is None else int(channel), _f(out))
    return out


def gauss_taps(sigma: float) -> np.ndarray:
    """The 2R+1 taps of the defocus kernel, R = ceil(3 sigma) [R31]."""
    w = np.zeros(257, np.float32)
    R = lib().evo_gauss_taps(float(sigma), _f(w), w.size)
    assert R >= 0, "sigma too large"
    return w[:2 * R + 1].copy()


def blur(frame: np.ndarray, taps: np.ndarray) -> np.ndarray:
    """Separable convolution of one [H,W] float32 frame with `taps` (rows, then columns; replicated border) [R31]."""
    frame = np.ascontiguousarray(frame, np.float32)
    H, W = frame.shape
    taps = np.ascontiguousarray(taps, np.float32)
    tmp, dst = np.empty((H, W), np.float32), np.empty((H, W), np.float32)
    lib().evo_blur(H, W, (taps.size - 1) // 2, _f(taps), _f(frame), _f(tmp), _f(dst))
    return dst


def splat(i: int, S: int, src_is_B: bool, disp: np.ndarray, Zsrc: np.ndarray, Zoth: np.ndarray
          ) -> np.ndarray:
    """Eq. 5-7 for one env, one direction, one substep.  Returns the z-buffer [H,W] uint64."""
    H, W = Zsrc.shape
    z = np.full((H, W), 0xFFFFFFFFFFFFFFFF, dtype=np.uint64)
    lib().evo_splat(H, W, i, S, int(src_is_B), _f(np.ascontiguousarray(disp, np.float32)),
                    _f(np.ascontiguousarray(Zsrc, np.float32)), _f(np.ascontiguousarray(Zoth, np.float32)),
                    _p(z, C.c_uint64))
    return z


def wsplat(i: int, S: int, src_is_B: bool, disp: np.ndarray, Zsrc: np.ndarray, Zoth: np.ndarray, Lsrc: np.ndarray,
           zbuf: np.ndarray) -> np.ndarray:
    """Weighted front-surface accumulation [R32] of one direction against its finished z-buffer ``zbuf`` (from
    ``splat``).  Returns acc [H,W,2] int64: (sum W L 2^24, sum W), W in units of 2^-20."""
    H, W = Zsrc.shape
    acc = np.zeros((H, W, 2), np.int64)
    lib().evo_wsplat(H, W, i, S, int(src_is_B), _f(np.ascontiguousarray(disp, np.float32)),
                     _f(np.ascontiguousarray(Zsrc, np.float32)), _f(np.ascontiguousarray(Zoth, np.float32)),
                     _f(np.ascontiguousarray(Lsrc, np.float32)), _p(np.ascontiguousarray(zbuf, np.uint64), C.c_uint64),
                     _p(acc, C.c_int64))
    return acc


def composite(i: int, S: int, mode: int, zA: np.ndarray, zB: np.ndarray, LA: np.ndarray, LB: np.ndarray,
              Lprev: np.ndarray):
    """The composite rule (R19) for one env and one substep from the two z-buffers [H,W] uint64 of
    ``splat`` and the log frames [H,W].  Returns (Lhat float32, dir uint8: 0 B / 1 A / 2 blend / 3 hole, idx uint32)."""
    H, W = zA.shape
    Lhat = np.empty((H, W), np.float32)
    d = np.empty((H, W), np.uint8)
    idx = np.empty((H, W), np.uint32)
    lib().evo_composite(H, W, i, S, int(mode), _p(np.ascontiguousarray(zA, np.uint64), C.c_uint64),
                        _p(np.ascontiguousarray(zB, np.uint64), C.c_uint64),
                        _f(np.ascontiguousarray(LA, np.float32)), _f(np.ascontiguousarray(LB, np.float32)),
                        _f(np.ascontiguousarray(Lprev, np.float32)), _f(Lhat), _p(d, C.c_uint8), _p(idx, C.c_uint32))
    return Lhat, d, idx


def event_frames(frames: np.ndarray, L0: np.ndarray, c_pos: float, c_neg: float, T: float,
                 Lref0: Optional[np.ndarray] = None, theta_on: Optional[np.ndarray] = None,
                 theta_off: Optional[np.ndarray] = None, tau_r: float = 0.0, t_last0: Optional[np.ndarray] = None,
                 noise: Optional[dict] = None):
    """Event stage alone (Eq. 4): feed a sequence of S log frames [S,H,W] to one env.
    theta_on / theta_off [H,W]: per-pixel thresholds replacing c_pos / c_neg (Eq. 8).
    tau_r > 0: refractory period; t_last0 [H,W] = stamps of the last emitted events relative to
    the start of these frames (default -inf); the final t_last is returned as a third value.

    Returns (events, Lref_final).  Lref and Lprev start at L0 (or Lref0 for the reference)."""
    frames = np.ascontiguousarray(frames, np.float32)
    S, H, W = frames.shape
    Lprev = np.ascontiguousarray(L0, np.float32).copy()
    Lref = Lprev.copy() if Lref0 is None else np.ascontiguousarray(Lref0, np.float32).copy()
    ton = None if theta_on is None else np.ascontiguousarray(theta_on, np.float32)
    toff = None if theta_off is None else np.ascontiguousarray(theta_off, np.float32)
    assert (ton is None) == (toff is None)
    nz, _hot = _noise_struct(noise, 0)
    tl0 = np.full((H, W), -np.inf, np.float32) if t_last0 is None else np.ascontiguousarray(t_last0, np.float32)
    cap = 1 << 16
    while True:
        ev = np.zeros(cap, dtype=EVENT_DTYPE)
        lr, lp = Lref.copy(), Lprev.copy()
        tl = tl0.copy()
        n = 0
        for i in range(1, S + 1):
            n += lib().evo_event_frame(H, W, 0, 0, i, S, float(T), float(c_pos), float(c_neg),
                                       _f(ton) if ton is not None else None, _f(toff) if toff is not None else None,
                                       float(tau_r), _f(tl), C.addressof(nz) if nz is not None else None,
                                       _f(frames[i - 1]), _f(lr), _f(lp), ev.ctypes.data, cap, n, None)
        if n <= cap:
            return (ev[:n], lr, tl) if tau_r > 0.0 else (ev[:n], lr)
        cap = int(n)


def _noise_struct(noise: Optional[dict], env: int):
    """noise = dict(seed, r_leak, r_shot, r_hot, i_white, eps, hot=None or uint8 [E,H,W] / [H,W]) -> (Noise, keepalive)."""
    if noise is None:
        return None, None
    hot = noise.get("hot")
    hp = None
    if hot is not None:
        hot = np.ascontiguousarray(hot, np.uint8)
        hp = np.ascontiguousarray(hot[env] if hot.ndim == 3 else hot)
    nz = Noise(int(noise["seed"]), float(noise.get("r_leak", 0.0)), float(noise.get("r_shot", 0.0)),
               float(noise.get("r_hot", 0.0)), float(noise.get("i_white", 1.0)), float(noise.get("eps", 1e-3)),
               hp.ctypes.data if hp is not None else None)
    return nz, hp


class Oracle:
    """Stateful oracle over E envs: ``step(keyframe)`` mirrors evis_step."""

    def __init__(self, num_envs: int, height: int, width: int, substeps: int, c_pos: float, c_neg: float,
                 log_eps: float, keyframe_dt: float, composite_mode: int = 0, debug: bool = False,
                 theta_on: Optional[np.ndarray] = None, theta_off: Optional[np.ndarray] = None,
                 tau_r: float = 0.0, margin: int = 0, channel: Optional[int] = None, noise: Optional[dict] = None,
                 defocus_sigma: Optional[float] = None):
        self.E, self.H, self.W, self.S = num_envs, height, width, substeps
        self.c_pos, self.c_neg, self.eps, self.T = c_pos, c_neg, log_eps, keyframe_dt
        self.mode = composite_mode
        # Eq. 8: per-pixel ON / OFF thresholds [E,H,W] replacing c_pos / c_neg (both or neither)
        assert (theta_on is None) == (theta_off is None)
        self.th_on = None if theta_on is None else np.ascontiguousarray(theta_on, np.float32).reshape(num_envs, height, width)
        self.th_off = None if theta_off is None else np.ascontiguousarray(theta_off, np.float32).reshape(num_envs, height, width)
        self.debug = debug
        # refractory period: stamps of the last emitted events, relative to the current interval
        # over-render margin (Supp. B): height x width is the over-rendered frame; the warp runs on
        # all of it, then `margin` pixels are cropped off each side: events outside the crop are dropped and the
        # others are reported in the cropped frame's coordinates [R27]
        self.noise = None if noise is None else dict(noise, eps=log_eps)   # Eq. 9-10 and hot pixels [R29]
        self.channel = channel                     # colour events: None = luminance, 0/1/2 = R/G/B
        self.margin = int(margin)
        assert 0 <= 2 * self.margin < min(height, width)
        # defocus [R31]: None = off; a sigma (>= 0) = the warped LINEAR frame of every substep is blurred
        self.taps = None if defocus_sigma is None else gauss_taps(defocus_sigma)
        assert self.taps is None or composite_mode == 0, "defocus is defined for the B-primary composite"
        assert composite_mode in (0, 1, 2)         # 2 = weighted front-surface splat [R32]
        self.Iprev = None
        self.tau_r = float(tau_r)
        self.t_last = np.full((num_envs, height, width), -np.inf, np.float32)
        self.calls = 0
        self.prev = None
        self.Lref = None
        self.Lprev = None
        self.holes = 0
        self.dbg: Dict[str, np.ndarray] = {}

    def step(self, rad, mv_bwd, depth, mv_fwd=None) -> np.ndarray:
        """Consume one keyframe.  The first call initialises (Lref = L, no events) [R6]; every later
        call returns the events of interval kf = call_index - 1 in (env, substep, y, x, k) order.
        ``mv_fwd`` is the forward field OF THIS keyframe, used when it plays the role of A in the
        NEXT call; None = reuse -mv_bwd."""
        E, H, W, S = self.E, self.H, self.W, self.S
        rad = np.ascontiguousarray(rad, np.float32).reshape(E, H, W, 3)
        mB = np.ascontiguousarray(mv_bwd, np.float32).reshape(E, H, W, 2)
        ZB = np.ascontiguousarray(depth, np.float32).reshape(E, H, W)
        LB = log_luminance(rad, self.eps, self.channel)
        fwd = -mB if mv_fwd is None else np.ascontiguousarray(mv_fwd, np.float32).reshape(E, H, W, 2)
        fwd = np.ascontiguousarray(fwd)
        cur = dict(L=LB, m=mB, Z=ZB, fwd=fwd)
        if self.taps is not None:
            cur["I"] = linear_luminance(rad, self.channel)
        if self.calls == 0:
            if self.taps is not None:                  # the event model's first frame is the blurred keyframe too
                self.Iprev = cur["I"].copy()
                LB0 = np.stack([np.log(blur(cur["I"][e], self.taps).astype(np.float64) + np.float64(np.float32(self.eps)))
                                for e in range(E)]).astype(np.float32)
                self.Lref, self.Lprev = LB0.copy(), LB0.copy()
                self.prev = cur
                self.calls = 1
                return np.zeros(0, dtype=EVENT_DTYPE)
            self.Lref = LB.copy()
            self.Lprev = LB.copy()
            self.prev = cur
            self.calls = 1
            return np.zeros(0, dtype=EVENT_DTYPE)
        A = self.prev
        kf = self.calls - 1
        P = H * W
        zA = np.empty(P, np.uint64)
        zB = np.empty(P, np.uint64)
        Lhat = np.empty(P, np.float32)
        if self.debug:
            self.dbg = dict(winA=np.empty((E, S, H, W), np.uint32), winB=np.empty((E, S, H, W), np.uint32),
                            dir=np.empty((E, S, H, W), np.uint8), idx=np.empty((E, S, H, W), np.uint32),
                            Lhat=np.empty((E, S, H, W), np.float32), dL=np.empty((E, S, H, W), np.float32))
        holes = C.c_int64(0)
        cap = max(1 << 16, 4 * E * P)
        while True:
            ev = np.zeros(cap, dtype=EVENT_DTYPE)
            Lref, Lprev = self.Lref.copy(), self.Lprev.copy()
            t_last = self.t_last.copy()
            Iprev = None if self.taps is None else self.Iprev.copy()
            btmp, bout = np.empty(P, np.float32), np.empty(P, np.float32)
            waA, waB = np.zeros(2 * P, np.int64), np.zeros(2 * P, np.int64)
            holes.value = 0
            n = 0
            for e in range(E):
                nz, _hot = _noise_struct(self.noise, e)
                d = self.dbg
                n += lib().evo_interval(
                    H, W, S, self.mode, e, kf, self.margin, float(self.T), float(self.c_pos), float(self.c_neg),
                    _f(self.th_on[e]) if self.th_on is not None else None,
                    _f(self.th_off[e]) if self.th_off is not None else None,
                    self.tau_r, _f(t_last[e]), C.addressof(nz) if nz is not None else None,
                    _f(A["L"][e]), _f(A["fwd"][e]), _f(A["Z"][e]), _f(LB[e]), _f(mB[e]), _f(ZB[e]),
                    _f(Lref[e]), _f(Lprev[e]), _p(zA, C.c_uint64), _p(zB, C.c_uint64), _f(Lhat),
                    ev.ctypes.data, cap, n,
                    _p(d["winA"][e], C.c_uint32) if d else None, _p(d["winB"][e], C.c_uint32) if d else None,
                    _p(d["dir"][e], C.c_uint8) if d else None, _p(d["idx"][e], C.c_uint32) if d else None,
                    _f(d["Lhat"][e]) if d else None, _f(d["dL"][e]) if d else None, C.byref(holes),
                    -1 if self.taps is None else (self.taps.size - 1) // 2,
                    _f(self.taps) if self.taps is not None else None,
                    _f(A["I"][e]) if self.taps is not None else None, _f(cur["I"][e]) if self.taps is not None else None,
                    _f(Iprev[e]) if self.taps is not None else None, float(self.eps), _f(btmp), _f(bout),
                    _p(waA, C.c_int64), _p(waB, C.c_int64))
            if n <= cap:
                break
            cap = int(n)
        self.Lref, self.Lprev, self.t_last = Lref, Lprev, t_last
        self.Iprev = Iprev
        self.holes = holes.value
        self.prev = cur
        self.calls += 1
        ev = ev[:n]
        if self.margin:
            M = self.margin
            keep = (ev["x"] >= M) & (ev["x"] < W - M) & (ev["y"] >= M) & (ev["y"] < H - M)
            ev = ev[keep].copy()
            ev["x"] -= M
            ev["y"] -= M
        return ev
