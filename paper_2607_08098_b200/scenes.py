"""Seeded analytic keyframe generator: the stand-in for the paper's RTX renderer.

The paper's renderer hands the interpolation stage, per keyframe, a scene-linear HDR colour
frame, a backward motion-vector map and a depth map (Sec. 3.3), anti-aliasing
disabled (Supp. A 311-315).  No renderer and no scene of the paper exists on this
box, so the workloads of BASELINE.json:configs are realised as point-sampled analytic scenes.

This module serves BOTH the CPU oracle tests and the CUDA path (it is the one module they may
share) and therefore holds NONE of the method's arithmetic: no luminance, no log, no warp, no
event model.  It only paints objects.

Determinism across devices: every per-object scalar (positions, velocities, cos/sin, 10^x, exp)
is computed on the host in Python floats; the per-pixel work uses only IEEE +, -, *, /, floor,
comparisons and integer bit operations in float64/int64 torch ops, one op per kernel (no fused
multiply-add), so the CPU and the CUDA device produce byte-identical keyframes.

Conventions: pixel (x, y) has its centre at integer coordinates, x right,
y down, motion vectors in pixels.  ``mv_bwd`` of keyframe k is the displacement from a pixel of
keyframe k to the position of the same surface point in keyframe k-1; ``mv_fwd``
is the displacement to its position in keyframe k+1.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Sequence, Tuple

import torch

_M64 = (1 << 64) - 1
BASE_SEED = 260708098


# ----------------------------------------------------------------------------------------------
# counter-based host RNG (splitmix64 finaliser over a packed key)
# ----------------------------------------------------------------------------------------------
def _mix64(z: int) -> int:
    z = (z + 0x9E3779B97F4A7C15) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def urand(seed: int, env: int, obj: int, fld: int) -> float:
    """U[0,1) keyed by (seed, env, object, field); 53 random bits."""
    z = _mix64(seed & _M64)
    z = _mix64(z ^ (env + 1))
    z = _mix64(z ^ ((obj + 1) << 20))
    z = _mix64(z ^ ((fld + 1) << 44))
    return (z >> 11) / float(1 << 53)


def _uni(seed, env, obj, fld, lo, hi):
    return lo + (hi - lo) * urand(seed, env, obj, fld)


# ----------------------------------------------------------------------------------------------
# workload description
# ----------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class SceneSpec:
    """One synthetic workload (shape + sensor parameters + scene recipe)."""
    name: str
    num_envs: int
    height: int
    width: int
    num_keyframes: int
    keyframe_dt: float          # T = 1/f_k  [s]
    substeps: int               # S (the paper's K)
    c_pos: float
    c_neg: float
    log_eps: float = 1e-3
    kind: str = "rects"         # "rects" | "disk" | "noise" (stress input, see _paint_noise)
    num_rects: int = 8
    v_max: float = 300.0        # rectangle velocity bound [px/s], per component
    ego_v_max: float = 0.0      # global translation bound [px/s], per component
    ramp_max: float = 0.0       # |rho| bound of the brightness ramp exp(rho t) [1/s]
    log10_rad: float = 2.0      # base radiance is 10^U[-log10_rad, +log10_rad]
    seed: int = BASE_SEED
    bg_textured: bool = False   # background plane carries a texture (needed when it moves)

    @property
    def pixels(self) -> int:
        return self.num_envs * self.height * self.width

    def max_motion_px(self) -> float:
        """Upper bound on |mv| (infinity norm) over the whole workload, in pixels."""
        if self.kind == "disk":
            r = 160.0
            return 2.0 * r * abs(math.sin(0.5 * 40.0 * self.keyframe_dt)) + 300.0 * self.keyframe_dt + 1.0
        return (self.v_max + self.ego_v_max) * self.keyframe_dt


def config(i: int) -> SceneSpec:
    """The workloads of BASELINE.json:configs, 1-based (configs[0] is ``config(1)``)."""
    if i == 1:
        return SceneSpec("cfg1_1env_346x260_S16", 1, 260, 346, 2, 1.0 / 60.0, 16, 0.2, 0.2,
                         num_rects=8, v_max=300.0, seed=BASE_SEED + 1)
    if i == 2:
        return SceneSpec("cfg2_16env_640x480_S16", 16, 480, 640, 61, 1.0 / 60.0, 16, 0.25, 0.25,
                         num_rects=32, v_max=600.0, seed=BASE_SEED + 2)
    if i == 3:
        return SceneSpec("cfg3_64env_1280x720_S33_disk", 64, 720, 1280, 31, 1.0 / 30.0, 33, 0.2, 0.3,
                         kind="disk", num_rects=0, v_max=300.0, log10_rad=3.0, seed=BASE_SEED + 3,
                         bg_textured=True)
    if i == 4:
        return SceneSpec("cfg4_256env_346x260_S16_rl", 256, 260, 346, 61, 1.0 / 60.0, 16, 0.2, 0.2,
                         num_rects=16, v_max=300.0, ego_v_max=800.0, ramp_max=1.0,
                         seed=BASE_SEED + 4, bg_textured=True)
    raise ValueError("config index must be 1..4 (config 5 is a sweep, see sweep_points())")


SWEEP_SHAPES = [(1, 1080, 1920), (16, 480, 640), (64, 260, 346), (256, 120, 160), (1024, 128, 128)]
SWEEP_SUBSTEPS = [8, 16, 33, 166]


def sweep_points() -> List[SceneSpec]:
    """BASELINE.json config 5: fixed total pixels, envs x resolution x S; scenes as config 1."""
    out = []
    for (e, h, w) in SWEEP_SHAPES:
        for s in SWEEP_SUBSTEPS:
            out.append(SceneSpec(f"cfg5_{e}env_{w}x{h}_S{s}", e, h, w, 3, 1.0 / 60.0, s, 0.2, 0.2,
                                 num_rects=8, v_max=300.0, seed=BASE_SEED + 5))
    return out


def small(spec: SceneSpec, **kw) -> SceneSpec:
    """A reduced copy of a workload (same recipe, smaller shape) for oracle-sized parity cases."""
    return replace(spec, **kw)


# ----------------------------------------------------------------------------------------------
# scene = per-object scalars, all computed on the host
# ----------------------------------------------------------------------------------------------
TEX_FLAT, TEX_CHECKER, TEX_NOISE = 0, 1, 2


@dataclass
class Obj:
    kind: int                  # 0 rectangle / plane, 1 disk
    depth: float
    x0: float                  # top-left corner (rect) or centre (disk) at t = 0
    y0: float
    w: float                   # size (rect) or radius (disk, in w)
    h: float
    vx: float                  # px/s (object + ego)
    vy: float
    tex: int
    cell: int                  # texture cell size [px]
    base: float                # base radiance
    tint: Sequence[float]      # 3 channel multipliers
    lo: float                  # texture low / high multipliers (10^(-a/2), 10^(+a/2))
    hi: float
    omega: float = 0.0         # disk angular rate [rad/s]
    spokes: int = 0            # disk: number of spoke pairs
    tex_id: int = 0


@dataclass
class Scene:
    spec: SceneSpec
    objs: List[List[Obj]]      # per env, sorted far -> near (painter's order)
    ramp: List[float]          # per env rho

    def time_of(self, k: int) -> float:
        return k * self.spec.keyframe_dt


def make_scene(spec: SceneSpec) -> Scene:
    H, W = spec.height, spec.width
    a_dec = 0.5  # texture contrast: half a decade between the two texture levels
    lo, hi = 10.0 ** (-a_dec / 2), 10.0 ** (a_dec / 2)
    all_objs, ramps = [], []
    for e in range(spec.num_envs):
        s = spec.seed
        egox = _uni(s, e, 1000, 0, -spec.ego_v_max, spec.ego_v_max) if spec.ego_v_max > 0 else 0.0
        egoy = _uni(s, e, 1000, 1, -spec.ego_v_max, spec.ego_v_max) if spec.ego_v_max > 0 else 0.0
        ramps.append(_uni(s, e, 1000, 2, -spec.ramp_max, spec.ramp_max) if spec.ramp_max > 0 else 0.0)
        objs: List[Obj] = []
        # background plane at 10 m: covers everything (huge rectangle), textured when it moves
        bg_vx, bg_vy = egox, egoy
        if spec.kind == "disk":
            bg_vx += _uni(s, e, 999, 3, -spec.v_max, spec.v_max)
            bg_vy += _uni(s, e, 999, 4, -spec.v_max, spec.v_max)
        bg_tex = TEX_NOISE if spec.bg_textured else TEX_FLAT
        objs.append(Obj(0, 10.0, -1.0e6, -1.0e6, 4.0e6, 4.0e6, bg_vx, bg_vy, bg_tex,
                        int(4 + math.floor(13 * urand(s, e, 999, 5))),
                        10.0 ** _uni(s, e, 999, 6, -spec.log10_rad, spec.log10_rad),
                        [_uni(s, e, 999, 7 + c, 0.5, 1.0) for c in range(3)], lo, hi, tex_id=999))
        for o in range(spec.num_rects):
            w = _uni(s, e, o, 0, 20.0, 120.0)
            h = _uni(s, e, o, 1, 20.0, 120.0)
            objs.append(Obj(0, _uni(s, e, o, 2, 1.0, 9.0),
                            _uni(s, e, o, 3, -0.25 * w, W - 0.75 * w), _uni(s, e, o, 4, -0.25 * h, H - 0.75 * h),
                            w, h,
                            _uni(s, e, o, 5, -spec.v_max, spec.v_max) + egox,
                            _uni(s, e, o, 6, -spec.v_max, spec.v_max) + egoy,
                            TEX_CHECKER if urand(s, e, o, 7) < 0.5 else TEX_NOISE,
                            int(4 + math.floor(13 * urand(s, e, o, 8))),
                            10.0 ** _uni(s, e, o, 9, -spec.log10_rad, spec.log10_rad),
                            [_uni(s, e, o, 10 + c, 0.5, 1.0) for c in range(3)], lo, hi, tex_id=o))
        if spec.kind == "disk":
            r = _uni(s, e, 500, 0, 100.0, 160.0)
            objs.append(Obj(1, 2.0, _uni(s, e, 500, 1, 0.3 * W, 0.7 * W), _uni(s, e, 500, 2, 0.3 * H, 0.7 * H),
                            r, r, 0.0, 0.0, TEX_FLAT, 8,
                            10.0 ** _uni(s, e, 500, 3, -spec.log10_rad, spec.log10_rad),
                            [_uni(s, e, 500, 4 + c, 0.5, 1.0) for c in range(3)], lo, hi,
                            omega=_uni(s, e, 500, 7, 5.0, 40.0) * (1.0 if urand(s, e, 500, 8) < 0.5 else -1.0),
                            spokes=int(4 + math.floor(9 * urand(s, e, 500, 9))), tex_id=500))
        objs.sort(key=lambda ob: -ob.depth)   # far -> near; python sort is stable
        all_objs.append(objs)
    return Scene(spec, all_objs, ramps)


# ----------------------------------------------------------------------------------------------
# per-pixel painting (torch, device-agnostic, float64 / int64 only)
# ----------------------------------------------------------------------------------------------
def _hash01(ix: torch.Tensor, iy: torch.Tensor, salt: int) -> torch.Tensor:
    """Integer cell hash -> [0,1) float64.  All products stay below 2^63 (no wrap needed)."""
    m32 = 0xFFFFFFFF
    h = ((ix & 0xFFFF) * 73856093) ^ ((iy & 0xFFFF) * 19349663) ^ ((salt & 0xFFFF) * 83492791)
    h = h & m32
    h = ((h ^ (h >> 16)) * 0x45D9F3B) & m32
    h = ((h ^ (h >> 16)) * 0x45D9F3B) & m32
    h = h ^ (h >> 16)
    return h.to(torch.float64) / 4294967296.0


def _col(vals, device) -> torch.Tensor:
    return torch.tensor(vals, device=device, dtype=torch.float64).view(-1, 1, 1)


def _paint_chunk(scene: Scene, t: float, t_prev: float, t_next: float, device, envs: Sequence[int],
                 want_mv: bool) -> Dict[str, torch.Tensor]:
    """Paint the listed envs at once: object slot by object slot (far -> near), vectorised over envs."""
    spec = scene.spec
    H, W = spec.height, spec.width
    f64 = torch.float64
    n = len(envs)
    ys = torch.arange(H, device=device, dtype=f64).view(1, H, 1)
    xs = torch.arange(W, device=device, dtype=f64).view(1, 1, W)
    rad = [torch.zeros((n, H, W), device=device, dtype=f64) for _ in range(3)]
    depth = torch.zeros((n, H, W), device=device, dtype=f64)
    mv = [torch.zeros((n, H, W), device=device, dtype=f64) for _ in range(4)]  # bwd x,y, fwd x,y
    gain = [math.exp(scene.ramp[e] * t) for e in envs]
    nslots = len(scene.objs[envs[0]])
    for slot in range(nslots):
        obs = [scene.objs[e][slot] for e in envs]
        is_disk = obs[0].kind == 1
        assert all((ob.kind == 1) == is_disk for ob in obs)
        px = [ob.x0 + ob.vx * t for ob in obs]
        py = [ob.y0 + ob.vy * t for ob in obs]
        u = xs - _col(px, device)
        v = ys - _col(py, device)
        if not is_disk:
            inside = (u >= 0.0) & (u < _col([ob.w for ob in obs], device)) \
                & (v >= 0.0) & (v < _col([ob.h for ob in obs], device))
            cell = _col([float(ob.cell) for ob in obs], device)
            cx = torch.floor(u / cell).to(torch.int64)
            cy = torch.floor(v / cell).to(torch.int64)
            salt = torch.tensor([ob.tex_id for ob in obs], device=device, dtype=torch.int64).view(-1, 1, 1)
            tex = torch.tensor([ob.tex for ob in obs], device=device, dtype=torch.int64).view(-1, 1, 1)
            par = ((cx + cy) & 1).to(f64)
            tau = torch.where(tex == TEX_CHECKER, par, _hash01(cx, cy, salt))
            lo = _col([ob.lo for ob in obs], device)
            hi = _col([ob.hi for ob in obs], device)
            lev = torch.where(tex == TEX_FLAT, torch.ones_like(tau), lo + (hi - lo) * tau)
            if want_mv:
                shape = (n, H, W)
                m = [_col([(ob.x0 + ob.vx * t_prev) - p_ for ob, p_ in zip(obs, px)], device).expand(shape),
                     _col([(ob.y0 + ob.vy * t_prev) - p_ for ob, p_ in zip(obs, py)], device).expand(shape),
                     _col([(ob.x0 + ob.vx * t_next) - p_ for ob, p_ in zip(obs, px)], device).expand(shape),
                     _col([(ob.y0 + ob.vy * t_next) - p_ for ob, p_ in zip(obs, py)], device).expand(shape)]
        else:
            rr = _col([ob.w * ob.w for ob in obs], device)
            inside = (u * u + v * v) <= rr
            # rotate into the disk frame by -theta(t): the spokes ride with the disk
            c = _col([math.cos(ob.omega * t) for ob in obs], device)
            s = _col([math.sin(ob.omega * t) for ob in obs], device)
            ur = c * u + s * v
            vr = c * v - s * u
            # sign of Im((ur + i vr)^m), m = spoke pairs: alternating sectors without atan2
            re, im = ur, vr
            mmax = max(ob.spokes for ob in obs)
            mcol = torch.tensor([ob.spokes for ob in obs], device=device, dtype=torch.int64).view(-1, 1, 1)
            sel = torch.where(mcol == 1, im, torch.zeros_like(im))
            for it in range(2, mmax + 1):
                re, im = re * ur - im * vr, re * vr + im * ur
                sel = torch.where(mcol == it, im, sel)
            lo = _col([ob.lo for ob in obs], device)
            hi = _col([ob.hi for ob in obs], device)
            lev = torch.where(sel > 0.0, hi.expand_as(sel), lo.expand_as(sel))
            if want_mv:
                ab = _col([math.cos(ob.omega * (t_prev - t)) for ob in obs], device)
                bb = _col([math.sin(ob.omega * (t_prev - t)) for ob in obs], device)
                af = _col([math.cos(ob.omega * (t_next - t)) for ob in obs], device)
                bf = _col([math.sin(ob.omega * (t_next - t)) for ob in obs], device)
                m = [(ab * u - bb * v) - u, (bb * u + ab * v) - v,
                     (af * u - bf * v) - u, (bf * u + af * v) - v]
        for ch in range(3):
            scale = _col([ob.base * ob.tint[ch] * g for ob, g in zip(obs, gain)], device)
            rad[ch] = torch.where(inside, lev * scale, rad[ch])
        depth = torch.where(inside, _col([ob.depth for ob in obs], device).expand_as(depth), depth)
        if want_mv:
            for q in range(4):
                mv[q] = torch.where(inside, m[q], mv[q])
    out = {"rad": torch.stack(rad, dim=-1).to(torch.float32).contiguous(),
           "depth": depth.to(torch.float32).contiguous()}
    if want_mv:
        out["mv_bwd"] = torch.stack(mv[0:2], dim=-1).to(torch.float32).contiguous()
        out["mv_fwd"] = torch.stack(mv[2:4], dim=-1).to(torch.float32).contiguous()
    return out


def _paint(scene: Scene, t: float, t_prev: float, t_next: float, device, envs: Sequence[int],
           want_mv: bool = True, max_chunk_px: int = 1 << 23) -> Dict[str, torch.Tensor]:
    per_env = scene.spec.height * scene.spec.width
    step = max(1, max_chunk_px // per_env)
    parts = [_paint_chunk(scene, t, t_prev, t_next, device, envs[i:i + step], want_mv)
             for i in range(0, len(envs), step)]
    if len(parts) == 1:
        return parts[0]
    return {k: torch.cat([p[k] for p in parts], dim=0) for k in parts[0]}


def _paint_noise(scene: Scene, k: int, device, envs: Sequence[int]) -> Dict[str, torch.Tensor]:
    """kind == "noise": a stress input, not a scene.  Every pixel of every keyframe gets hashed radiance,
    hashed motion vectors in [-v_max T, v_max T) (quantised to 1/4 px, so integer and half-integer
    landings and therefore every footprint class occur) and a depth drawn from eight values (so depth
    ties are everywhere).  Keyframes are unrelated to each other: it exercises the z-test, the tie-break,
    hole filling and the event model under conflicts no rendered scene produces."""
    spec = scene.spec
    H, W = spec.height, spec.width
    M = spec.v_max * spec.keyframe_dt
    ys = torch.arange(H, device=device, dtype=torch.int64).view(1, H, 1)
    xs = torch.arange(W, device=device, dtype=torch.int64).view(1, 1, W)
    es = torch.tensor(list(envs), device=device, dtype=torch.int64).view(-1, 1, 1)
    salt0 = (spec.seed & 0xFFF) * 131 + k * 17

    def h(field):
        return _hash01(xs + 7 * field + 1000 * es, ys + 13 * k, torch.full_like(es, salt0 + 31 * field))

    rad = torch.stack([10.0 ** (spec.log10_rad * (2.0 * h(c) - 1.0)) for c in range(3)], dim=-1)
    q = 4.0
    mv = [torch.floor((2.0 * h(3 + c) - 1.0) * M * q) / q for c in range(4)]
    still = h(9) < 0.25                                    # a quarter of the pixels rest
    mv = [torch.where(still, torch.zeros_like(m), m) for m in mv]
    depth = 1.0 + torch.floor(8.0 * h(8))
    return {"rad": rad.to(torch.float32).contiguous(), "depth": depth.to(torch.float32).contiguous(),
            "mv_bwd": torch.stack(mv[0:2], dim=-1).to(torch.float32).contiguous(),
            "mv_fwd": torch.stack(mv[2:4], dim=-1).to(torch.float32).contiguous()}


def threshold_maps(spec: SceneSpec, sigma: float = 0.03, theta_min: float = 0.01, device="cpu"
                   ) -> Tuple[torch.Tensor, torch.Tensor]:
    """Seeded per-pixel ON / OFF threshold maps [E,H,W] float32 for evis_set_thresholds: the draw the paper
    states for threshold mismatch, theta ~ max(N(C, sigma^2), theta_min), once per pixel (PAPER.md:137-142,
    Eq. 8).  Input synthesis only (the method's arithmetic is not here): Box-Muller on the counter hash of
    (pixel, salt), in float64 on the CPU so that the maps do not depend on the device."""
    E, H, W = spec.num_envs, spec.height, spec.width
    iy, ix = torch.meshgrid(torch.arange(E * H, dtype=torch.int64), torch.arange(W, dtype=torch.int64), indexing="ij")
    out = []
    for salt, c in ((0x51ED + spec.seed, spec.c_pos), (0xA7C3 + spec.seed, spec.c_neg)):
        u1 = _hash01(ix, iy, salt).double().clamp_min(1e-12)
        u2 = _hash01(ix, iy, salt + 1).double()
        n = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)
        theta = torch.clamp(c + sigma * n, min=theta_min).float().reshape(E, H, W).contiguous()
        out.append(theta.to(device))
    return out[0], out[1]


def render_keyframe(scene: Scene, k: int, device="cpu", envs: Optional[Sequence[int]] = None
                    ) -> Dict[str, torch.Tensor]:
    """Keyframe k: ``rad[E,H,W,3]``, ``mv_bwd[E,H,W,2]``, ``mv_fwd[E,H,W,2]``, ``depth[E,H,W]`` (float32)."""
    T = scene.spec.keyframe_dt
    envs = list(range(scene.spec.num_envs)) if envs is None else list(envs)
    if scene.spec.kind == "noise":
        return _paint_noise(scene, k, torch.device(device), envs)
    return _paint(scene, k * T, (k - 1) * T, (k + 1) * T, torch.device(device), envs)


def render_at(scene: Scene, t: float, device="cpu", envs: Optional[Sequence[int]] = None
              ) -> Dict[str, torch.Tensor]:
    """Ground-truth radiance and depth at an arbitrary time t (no motion vectors)."""
    envs = list(range(scene.spec.num_envs)) if envs is None else list(envs)
    return _paint(scene, t, t, t, torch.device(device), envs, want_mv=False)
