"""Pins for the CPU oracle (oracle/evis_oracle.c): it is checked against what the paper and the
mathematics fix -- printed constants, closed forms, invariants, special cases and brute force --
never against itself.  CPU only.  Pin numbers follow SURVEY.md Sec. 8(c) / DESIGN.md.
"""
import math
import os

import numpy as np
import pytest

from oracle import evis_oracle as orc
from paper_2607_08098_b200 import scenes

GOLD = os.path.join(os.path.dirname(__file__), "golden")
EMPTY = np.uint64(0xFFFFFFFFFFFFFFFF)


def _rng(seed):
    return np.random.default_rng(seed)


# ------------------------------------------------------------------------------------------------
# Eq. 3 + log
# ------------------------------------------------------------------------------------------------
def test_rec709_weights_and_log_closed_forms():
    """PAPER.md:96 prints the weights; L = log(I + eps).  Single-channel inputs
    isolate each weight (a permuted weight fails), math.log is the independent library routine."""
    w = {}
    for line in open(os.path.join(GOLD, "rec709_weights.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        w[k] = float(v)
    assert abs(w["R"] + w["G"] + w["B"] - 1.0) < 1e-12
    eps = 1e-3
    rad = np.array([[1, 0, 0], [0, 1, 0], [0, 0, 1], [1, 1, 1], [0, 0, 0], [2.5, 0.5, 4.0],
                    [-1.0, 0.0, 0.0]], dtype=np.float32)
    L = orc.log_luminance(rad, eps)
    e32 = float(np.float32(eps))
    exp = [math.log(w["R"] + e32), math.log(w["G"] + e32), math.log(w["B"] + e32),
           math.log(w["R"] + w["G"] + w["B"] + e32), math.log(e32),
           math.log(2.5 * w["R"] + 0.5 * w["G"] + 4.0 * w["B"] + e32),
           math.log(e32)]                      # negative luminance clamps to 0 (reading R3)
    for got, want in zip(L, exp):
        assert got == np.float32(want) or abs(float(got) - want) <= 2.0 ** -23 * abs(want)


def test_log_is_natural_log_of_linear_radiance():
    """exp(L) - eps recovers I: pins log base e (R1) against a wrong base and a missing eps."""
    r = _rng(1)
    rad = (10.0 ** r.uniform(-3, 3, size=(1000, 3))).astype(np.float32)
    L = orc.log_luminance(rad, 1e-3).astype(np.float64)
    I = 0.2126 * rad[:, 0].astype(np.float64) + 0.7152 * rad[:, 1] + 0.0722 * rad[:, 2]
    assert np.allclose(np.exp(L) - np.float32(1e-3), I, rtol=2e-6, atol=1e-8)  # L is rounded to binary32


# ------------------------------------------------------------------------------------------------
# helpers to drive the warp on hand-made keyframes
# ------------------------------------------------------------------------------------------------
def _oracle(E, H, W, S, c=0.2, mode=0, T=1.0 / 60, eps=1e-3, cn=None):
    return orc.Oracle(E, H, W, S, c, c if cn is None else cn, eps, T, composite_mode=mode, debug=True)


def _rad_from_L(L, eps=1e-3):
    """Grey radiance whose log-luminance is (close to) L: only used to feed Oracle.step."""
    I = np.exp(L.astype(np.float64)) - eps
    return np.repeat(I[..., None], 3, axis=-1).astype(np.float32)


# ------------------------------------------------------------------------------------------------
# P1: zero motion, A = B
# ------------------------------------------------------------------------------------------------
def test_p1_zero_motion_is_identity_and_static_scene_is_silent():
    r = _rng(2)
    H, W, S = 13, 17, 5
    rad = (10.0 ** r.uniform(-2, 2, size=(1, H, W, 3))).astype(np.float32)
    depth = r.uniform(1, 9, size=(1, H, W)).astype(np.float32)
    mv = np.zeros((1, H, W, 2), np.float32)
    o = _oracle(1, H, W, S)
    assert len(o.step(rad, mv, depth)) == 0
    ev = o.step(rad, mv, depth)
    own = np.arange(H * W, dtype=np.uint32).reshape(H, W)
    L = orc.log_luminance(rad, 1e-3)[0]
    for i in range(S):
        assert np.array_equal(o.dbg["winA"][0, i], own)
        assert np.array_equal(o.dbg["winB"][0, i], own)
        assert np.array_equal(o.dbg["dir"][0, i], np.zeros((H, W), np.uint8))   # B is primary
        assert np.array_equal(o.dbg["Lhat"][0, i], L)
    assert len(ev) == 0 and o.holes == 0


# ------------------------------------------------------------------------------------------------
# P2: f = 1 reproduces keyframe B for ANY motion field (Eq. 5: q_B = p at f = 1)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", [0])
def test_p2_last_substep_reproduces_keyframe_b(mode):
    r = _rng(3)
    H, W, S = 16, 21, 7
    o = _oracle(1, H, W, S, mode=mode)
    for _ in range(3):
        rad = (10.0 ** r.uniform(-2, 2, size=(1, H, W, 3))).astype(np.float32)
        depth = r.uniform(0.5, 9, size=(1, H, W)).astype(np.float32)
        mv = r.uniform(-6, 6, size=(1, H, W, 2)).astype(np.float32)
        o.step(rad, mv, depth)
    own = np.arange(H * W, dtype=np.uint32).reshape(H, W)
    assert np.array_equal(o.dbg["winB"][0, S - 1], own)
    assert np.array_equal(o.dbg["Lhat"][0, S - 1], orc.log_luminance(rad, 1e-3)[0])
    assert np.array_equal(o.Lprev[0], orc.log_luminance(rad, 1e-3)[0])


# ------------------------------------------------------------------------------------------------
# P3: integer-pixel translation warps exactly (signs of Eq. 5 in both directions, A-fill)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("d", [(1, 0), (-2, 1), (0, -1), (3, 2)])
def test_p3_integer_translation_warps_exactly(d):
    H, W, S = 20, 24, 4                      # S a power of two: i/S exact in binary32
    dx, dy = d
    r = _rng(4)
    big = r.uniform(-3, 3, size=(H + 64, W + 64)).astype(np.float32)   # texture on an infinite plane

    def tex(px, py):                          # log value of the surface point under pixel (x,y)
        ys, xs = np.mgrid[0:H, 0:W]
        return big[ys - py + 32, xs - px + 32]

    LA, LB = tex(0, 0), tex(S * dx, S * dy)   # surface moved by D = S d between the keyframes
    mv = np.empty((1, H, W, 2), np.float32)
    mv[..., 0], mv[..., 1] = -S * dx, -S * dy            # backward MV: where it was in A
    depth = np.full((1, H, W), 3.0, np.float32)
    z64 = {}
    for i in range(1, S + 1):
        zA = orc.splat(i, S, False, -mv[0], depth[0], depth[0])
        zB = orc.splat(i, S, True, mv[0], depth[0], depth[0])
        z64[i] = (zA, zB)
        want = tex(i * dx, i * dy)
        ys, xs = np.mgrid[0:H, 0:W]
        # B covers q iff its source q + (S-i) d lies inside; A iff q - i d lies inside
        sbx, sby = xs + (S - i) * dx, ys + (S - i) * dy
        sax, say = xs - i * dx, ys - i * dy
        inB = (sbx >= 0) & (sbx < W) & (sby >= 0) & (sby < H)
        inA = (sax >= 0) & (sax < W) & (say >= 0) & (say < H)
        assert np.array_equal(zB != EMPTY, inB)
        assert np.array_equal(zA != EMPTY, inA)
        assert np.array_equal((zB & np.uint64(0xFFFFFFFF))[inB], (sby * W + sbx)[inB].astype(np.uint64))
        assert np.array_equal((zA & np.uint64(0xFFFFFFFF))[inA], (say * W + sax)[inA].astype(np.uint64))
        got = np.where(inB, LB.ravel()[np.clip(sby * W + sbx, 0, H * W - 1)],
                       LA.ravel()[np.clip(say * W + sax, 0, H * W - 1)])
        assert np.array_equal(got[inA | inB], want[inA | inB])


def test_p3b_composite_through_the_full_interval():
    """Same translation, driven through Oracle.step: Lhat equals the analytic frame wherever either
    keyframe sees the surface; the rest are holes that hold the previous value."""
    H, W, S, dx, dy = 18, 22, 4, 2, -1
    r = _rng(5)
    big = r.uniform(-3, 3, size=(H + 64, W + 64)).astype(np.float32)
    ys, xs = np.mgrid[0:H, 0:W]
    tex = lambda px, py: big[ys - py + 32, xs - px + 32]
    o = _oracle(1, H, W, S)
    mv = np.empty((1, H, W, 2), np.float32)
    mv[..., 0], mv[..., 1] = -S * dx, -S * dy
    depth = np.full((1, H, W), 3.0, np.float32)
    radA, radB = _rad_from_L(tex(0, 0))[None], _rad_from_L(tex(S * dx, S * dy))[None]
    LA, LB = orc.log_luminance(radA, 1e-3)[0], orc.log_luminance(radB, 1e-3)[0]
    o.step(radA, mv, depth)
    o.step(radB, mv, depth)
    prev = LA
    for i in range(1, S + 1):
        sbx, sby = xs + (S - i) * dx, ys + (S - i) * dy
        sax, say = xs - i * dx, ys - i * dy
        inB = (sbx >= 0) & (sbx < W) & (sby >= 0) & (sby < H)
        inA = (sax >= 0) & (sax < W) & (say >= 0) & (say < H)
        want = np.where(inB, LB.ravel()[np.clip(sby * W + sbx, 0, H * W - 1)],
                        np.where(inA, LA.ravel()[np.clip(say * W + sax, 0, H * W - 1)], prev))
        assert np.array_equal(o.dbg["Lhat"][0, i - 1], want)
        assert np.array_equal(o.dbg["dir"][0, i - 1], np.where(inB, 0, np.where(inA, 1, 3)))
        prev = want


# ------------------------------------------------------------------------------------------------
# P16: composite mode 1 (R19): nearest of the two winners; the time-weighted blend where both hit the same surface
# ------------------------------------------------------------------------------------------------
def _key(z, idx):
    return (np.uint64(np.float32(z).view(np.uint32)) << np.uint64(32)) | np.uint64(idx)


def test_p16_blend_mode_by_hand():
    """Hand-made z-buffers of a 1 x 8 row, dyadic log values, S = 4 (f = i/4 exact): every case of the rule.
    Expected values are written out from R19, not computed by the rule's code:
      both hit, |Z_A - Z_B| <= 0.01 min  ->  (1 - f) L_A* + f L_B*      (swapped weights fail: L_A* != L_B*)
      both hit, depths apart             ->  the nearer one, from either side
      one hit -> it;  none -> the previous value.
    The 1 % boundary is inclusive: Z = 100 and 101 differ by exactly 0.01f * 100 = 1 in binary32."""
    S = 4
    assert np.float32(0.01) * np.float32(100.0) == np.float32(1.0)      # the boundary case is exact
    LA = np.array([[-2.0, 1.5, 0.25, 3.0, -1.0, 0.5, 2.0, -3.0]], np.float32)
    LB = np.array([[4.0, -0.5, 1.0, -2.0, 0.75, -1.5, 1.0, 2.5]], np.float32)
    Lprev = np.full((1, 8), 7.0, np.float32)
    E_ = EMPTY
    #             same depth   1% apart(incl)  just over 1%        A nearer       B nearer      only A   only B   none
    zA = np.array([[_key(2.0, 1), _key(100.0, 0), _key(100.0, 3), _key(1.0, 5), _key(8.0, 2), _key(3.0, 7), E_, E_]], np.uint64)
    zB = np.array([[_key(2.0, 6), _key(101.0, 4), _key(np.nextafter(np.float32(101.0), np.float32(200.0)), 4),
                    _key(4.0, 0), _key(2.0, 7), E_, _key(5.0, 3), E_]], np.uint64)
    for i in range(1, S + 1):
        f = i / S
        lh, d, idx = orc.composite(i, S, 1, zA, zB, LA, LB, Lprev)
        want = [(1 - f) * 1.5 + f * 1.0,          # LA[1], LB[6]
                (1 - f) * -2.0 + f * 0.75,        # LA[0], LB[4]   (boundary: still the same surface)
                3.0,                              # A at 100 is nearer than B at 101.00001: LA[3]
                0.5,                              # LA[5]
                2.5,                              # LB[7]
                -3.0,                             # LA[7]
                -2.0,                             # LB[3]
                7.0]                              # hold
        assert lh[0].tolist() == want, (i, lh[0].tolist())
        assert d[0].tolist() == [2, 2, 1, 1, 0, 1, 0, 3]
        assert idx[0].tolist() == [6, 4, 3, 5, 7, 7, 3, orc.NONE]
    # mode 0 on the same buffers: B wherever it hit, else A
    lh, d, _ = orc.composite(2, S, 0, zA, zB, LA, LB, Lprev)
    assert lh[0].tolist() == [1.0, 0.75, 0.75, 4.0, 2.5, -3.0, -2.0, 7.0]
    assert d[0].tolist() == [0, 0, 0, 0, 0, 1, 0, 3]


@pytest.mark.parametrize("d", [(1, 0), (-2, 1)])
def test_p16b_blend_is_a_linear_ramp_in_time_along_a_translation(d):
    """A plane translating by an integer d per substep whose brightness rises by delta between the keyframes:
    where both keyframes see the surface, mode 1 gives L_A(surface) + f delta -- the time-weighted blend of
    north_star, exact for dyadic values; the strip only B (only A) sees takes that keyframe's value; the rest
    holds.  The z-buffers come from evo_splat, pinned by P3 on this very scene.
    (P2 does not carry over to mode 1: at i = S direction A lands with Z = Z_B of its far end, so a nearer A
    surface may legitimately replace keyframe B's own pixel.)"""
    H, W, S = 20, 24, 4
    dx, dy = d
    r = _rng(16)
    big = (r.integers(-24, 25, size=(H + 64, W + 64)) / 8.0).astype(np.float32)     # dyadic texture
    ys, xs = np.mgrid[0:H, 0:W]
    tex = lambda px, py: big[ys - py + 32, xs - px + 32]
    delta = np.float32(0.75)
    LA, LB = tex(0, 0), tex(S * dx, S * dy) + delta
    mv = np.empty((H, W, 2), np.float32)
    mv[..., 0], mv[..., 1] = -S * dx, -S * dy
    Z = np.full((H, W), 3.0, np.float32)
    prev = LA.copy()
    for i in range(1, S + 1):
        f = i / S
        zA = orc.splat(i, S, False, -mv, Z, Z)
        zB = orc.splat(i, S, True, mv, Z, Z)
        lh, dirs, _ = orc.composite(i, S, 1, zA, zB, LA, LB, prev)
        sbx, sby = xs + (S - i) * dx, ys + (S - i) * dy
        sax, say = xs - i * dx, ys - i * dy
        inB = (sbx >= 0) & (sbx < W) & (sby >= 0) & (sby < H)
        inA = (sax >= 0) & (sax < W) & (say >= 0) & (say < H)
        surf = tex(i * dx, i * dy)                                      # the plane at time f, brightness of A
        want = np.where(inA & inB, surf + np.float32(f) * delta,
                        np.where(inB, surf + delta, np.where(inA, surf, prev)))
        assert np.array_equal(lh, want.astype(np.float32)), i
        assert np.array_equal(dirs, np.where(inA & inB, 2, np.where(inB, 0, np.where(inA, 1, 3))))
        prev = lh


# ------------------------------------------------------------------------------------------------
# P4: 8x8 brute force, gather form, straight from the definition of S(q) (Eq. 6)
# ------------------------------------------------------------------------------------------------
def _brute_winner(H, W, i, S, src_is_B, disp, Zsrc, Zoth):
    """For every target enumerate all sources; a source covers the target iff its landing point is
    strictly within 1 px of it in x and in y (positive bilinear weight); lexicographic min of
    (Zt, source index).  Inputs are dyadic so every product / sum below is exact in float64."""
    f = i / S
    w = (1 - f) if src_is_B else f
    out = np.full((H, W), -1, dtype=np.int64)
    for ty in range(H):
        for tx in range(W):
            best = None
            for sy in range(H):
                for sx in range(W):
                    dx, dy = float(disp[sy, sx, 0]), float(disp[sy, sx, 1])
                    qx, qy = sx + w * dx, sy + w * dy
                    if not (abs(qx - tx) < 1 and abs(qy - ty) < 1):
                        continue
                    jx, jy = math.floor(sx + dx + 0.5), math.floor(sy + dy + 0.5)
                    zs = float(Zsrc[sy, sx])
                    zo = float(Zoth[jy, jx]) if (0 <= jx < W and 0 <= jy < H) else zs
                    za, zb = (zo, zs) if src_is_B else (zs, zo)
                    zt = (1 - f) * za + f * zb
                    cand = (zt, sy * W + sx)
                    if best is None or cand < best:
                        best = cand
            if best is not None:
                out[ty, tx] = best[1]
    return out


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_p4_bruteforce_splat_winners_8x8(seed):
    H = W = 8
    S = 4
    r = _rng(100 + seed)
    levels = np.array([1.0, 1.5, 2.0, 3.0, 6.0], np.float32)       # many depth ties
    for src_is_B in (True, False):
        disp = (r.integers(-12, 13, size=(H, W, 2)) / 4.0).astype(np.float32)   # multiples of 1/4 px
        Zsrc = levels[r.integers(0, len(levels), size=(H, W))]
        Zoth = levels[r.integers(0, len(levels), size=(H, W))]
        for i in range(1, S + 1):
            z = orc.splat(i, S, src_is_B, disp, Zsrc, Zoth)
            got = np.where(z == EMPTY, -1, (z & np.uint64(0xFFFFFFFF)).astype(np.int64))
            want = _brute_winner(H, W, i, S, src_is_B, disp, Zsrc, Zoth)
            assert np.array_equal(got, want), (seed, src_is_B, i)


def test_p4b_interpolated_depth_is_eq7():
    """One source, different depth in A and B: the stored key carries (1-f) Z_A + f Z_B."""
    H = W = 4
    S = 4
    Zb = np.full((H, W), 2.0, np.float32)
    Za = np.full((H, W), 6.0, np.float32)
    disp = np.zeros((H, W, 2), np.float32)
    for i in range(1, S + 1):
        z = orc.splat(i, S, True, disp, Zb, Za)
        zt = (z >> np.uint64(32)).astype(np.uint32).view(np.float32)
        assert np.all(zt == np.float32((1 - i / S) * 6.0 + (i / S) * 2.0))
        z = orc.splat(i, S, False, disp, Za, Zb)     # direction A: source depth is Z_A
        zt = (z >> np.uint64(32)).astype(np.uint32).view(np.float32)
        assert np.all(zt == np.float32((1 - i / S) * 6.0 + (i / S) * 2.0))


def test_tie_break_gives_ceil_shift():
    """tests/golden/tie_break_ceil.txt (derivation there): constant-depth row shifted by delta."""
    H, W = 1, 32
    Z = np.full((H, W), 2.0, np.float32)
    for line in open(os.path.join(GOLD, "tie_break_ceil.txt")):
        if line.startswith("#") or not line.strip():
            continue
        delta, shift = float(line.split()[0]), int(line.split()[1])
        disp = np.zeros((H, W, 2), np.float32)
        disp[..., 0] = delta
        z = orc.splat(4, 4, False, disp, Z, Z)           # direction A at f = 1: q = p + delta
        idx = (z & np.uint64(0xFFFFFFFF)).astype(np.int64)[0]
        for t in range(W):
            src = t - shift
            if 0 <= src < W:
                assert z[0, t] != EMPTY and idx[t] == src, (delta, t)


# ------------------------------------------------------------------------------------------------
# P5: two overlapping rectangles at different depths: nearest wins, compare with the analytic render
# ------------------------------------------------------------------------------------------------
def test_p5_occlusion_matches_analytic_render():
    spec = scenes.SceneSpec("p5", 1, 64, 80, 2, 1.0 / 60.0, 8, 0.2, 0.2)
    lo = hi = 1.0
    mk = lambda depth, x0, y0, w, h, vx, vy, base, tid: scenes.Obj(
        0, depth, x0, y0, w, h, vx, vy, scenes.TEX_FLAT, 8, base, [1.0, 1.0, 1.0], lo, hi, tex_id=tid)
    objs = [mk(10.0, -1e6, -1e6, 4e6, 4e6, 0.0, 0.0, 0.05, 0),
            mk(6.0, 10.0, 12.0, 40.0, 30.0, 200.0, -90.0, 1.0, 1),      # far rectangle
            mk(2.0, 40.0, 20.0, 25.0, 28.0, -260.0, 120.0, 20.0, 2)]    # near rectangle crosses it
    sc = scenes.Scene(spec, [objs], [0.0])
    k0 = scenes.render_keyframe(sc, 0)
    k1 = scenes.render_keyframe(sc, 1)
    o = _oracle(1, spec.height, spec.width, spec.substeps)
    o.step(k0["rad"].numpy(), k0["mv_bwd"].numpy(), k0["depth"].numpy(), k0["mv_fwd"].numpy())
    o.step(k1["rad"].numpy(), k1["mv_bwd"].numpy(), k1["depth"].numpy(), k1["mv_fwd"].numpy())
    S, T = spec.substeps, spec.keyframe_dt
    worst = 1.0
    for i in range(1, S + 1):
        gt = scenes.render_at(sc, (i / S) * T)
        Lgt = orc.log_luminance(gt["rad"].numpy(), 1e-3)[0]
        got = o.dbg["Lhat"][0, i - 1]
        bad = got != Lgt
        # every disagreement must sit within 2 px of a depth silhouette of the true frame
        d = gt["depth"].numpy()[0]
        edge = np.zeros_like(bad)
        for sy in range(-2, 3):
            for sx in range(-2, 3):
                sh = np.roll(np.roll(d, sy, 0), sx, 1)
                edge |= sh != d
        assert not np.any(bad & ~edge), f"substep {i}: mismatch away from silhouettes"
        worst = min(worst, 1.0 - bad.mean())
    assert worst > 0.97
    # where both rectangles overlap in the true frame the near one (base 20) is what is seen
    gt = scenes.render_at(sc, 0.5 * T)
    assert o.holes < 0.02 * S * spec.height * spec.width


# ------------------------------------------------------------------------------------------------
# event stage alone: P6-P10 + hand-worked fixture
# ------------------------------------------------------------------------------------------------
def test_event_model_hand_worked_fixture():
    frames, evs, lref = [], [], None
    for line in open(os.path.join(GOLD, "event_model_by_hand.txt")):
        if line.startswith("frames"):
            frames = [float(v) for v in line.split()[1:]]
        elif line.startswith("events"):
            _, i, p, t = line.split()
            evs.append((int(i), int(p), float(t)))
        elif line.startswith("lref_final"):
            lref = float(line.split()[1])
    fr = np.array(frames, np.float32).reshape(len(frames), 1, 1)
    ev, lr = orc.event_frames(fr, np.array([[1.0]], np.float32), 0.25, 0.5, 1.0)
    assert [(int(e["substep"]), int(e["p"])) for e in ev] == [(i, p) for i, p, _ in evs]
    assert np.allclose([e["t_off"] for e in ev], [t for _, _, t in evs], atol=1e-12)
    assert float(lr[0, 0]) == lref


@pytest.mark.parametrize("splits", [1, 2, 5, 16, 33])
def test_p6_monotone_total_is_independent_of_substep_split(splits):
    """Monotone L: total count = floor(|L_end - L_0| / C) however the path is cut (Eq. 4 + update).
    Dyadic C and endpoints keep binary32 exact so the closed form is exact."""
    C = 0.125
    L0 = np.float32(-1.0)
    for total in (0.0625, 0.125, 0.9375, 3.0, 5.4375):
        for sign in (+1, -1):
            Lend = L0 + np.float32(sign * total)
            frames = (L0 + (Lend - L0) * (np.arange(1, splits + 1, dtype=np.float64) / splits))
            frames = frames.astype(np.float32).reshape(splits, 1, 1)
            frames[-1] = Lend
            ev, lr = orc.event_frames(frames, np.array([[L0]], np.float32), C, C, 1.0)
            assert len(ev) == math.floor(total / C)
            assert all(int(e["p"]) == sign for e in ev)


def test_p6b_ramp_of_k_plus_half_thresholds_gives_k_events():
    C = 0.2
    for k in range(0, 12):
        for sign in (+1, -1):
            frames = np.array([sign * (k + 0.5) * C], np.float32).reshape(1, 1, 1)
            ev, lr = orc.event_frames(frames, np.zeros((1, 1), np.float32), C, C, 1.0)
            assert len(ev) == k and all(int(e["p"]) == sign for e in ev)


def test_p7_residual_bounds_and_reconstruction():
    r = _rng(7)
    S, H, W = 40, 6, 7
    cp, cn = 0.2, 0.3
    frames = np.cumsum(r.normal(0, 0.4, size=(S, H, W)), axis=0).astype(np.float32)
    L0 = np.zeros((H, W), np.float32)
    lref, lprev = L0.copy(), L0.copy()
    npos = np.zeros((H, W), int)
    nneg = np.zeros((H, W), int)
    for i in range(S):
        ev, lref = orc.event_frames(frames[i:i + 1], lprev, cp, cn, 1.0, Lref0=lref)
        lprev = frames[i]
        d = frames[i] - lref
        assert np.all(d < cp + 1e-5) and np.all(d > -cn - 1e-5)       # sub-threshold residual kept
        for e in ev:
            (npos if e["p"] > 0 else nneg)[e["y"], e["x"]] += 1
    recon = L0 + cp * npos - cn * nneg
    assert np.all(np.abs(frames[-1] - recon) < max(cp, cn) + 1e-4)
    assert np.allclose(lref, recon, atol=1e-4)


def test_p8_linear_ramp_timestamps():
    """L(t) = r t sampled at S frames: k-th event at t = k C / r (timestamps linear in L, R8)."""
    C, r, S, T = 0.2, 37.0, 16, 1.0 / 60.0
    frames = np.array([r * (i / S) * T for i in range(1, S + 1)], np.float32).reshape(S, 1, 1)
    ev, _ = orc.event_frames(frames, np.zeros((1, 1), np.float32), C, C, T)
    n = math.floor(r * T / C)
    assert len(ev) == n
    for k, e in enumerate(ev, start=1):
        assert abs(e["t_off"] - k * np.float32(C) / r) < 2e-8


def test_p9_timestamps_ordered_and_inside_their_substep():
    r = _rng(9)
    S, H, W, T = 12, 5, 5, 1.0 / 30.0
    frames = np.cumsum(r.normal(0, 0.5, size=(S, H, W)), axis=0).astype(np.float32)
    ev, _ = orc.event_frames(frames, np.zeros((H, W), np.float32), 0.2, 0.3, T)
    assert len(ev) > 100
    dt = T / S
    last = {}
    for e in ev:
        i = int(e["substep"])
        assert (i - 1) * dt - 1e-12 <= e["t_off"] <= i * dt + 1e-12
        key = (int(e["x"]), int(e["y"]))
        assert e["t_off"] >= last.get(key, -1.0)
        last[key] = e["t_off"]


def test_p10_up_then_down_with_asymmetric_thresholds():
    cp, cn = 0.25, 0.5
    D = np.float32(1.1875)                       # dyadic: 4 ON events, residual 0.1875
    frames = np.array([D, 0.0], np.float32).reshape(2, 1, 1)
    ev, lr = orc.event_frames(frames, np.zeros((1, 1), np.float32), cp, cn, 1.0)
    on = [e for e in ev if e["p"] > 0]
    off = [e for e in ev if e["p"] < 0]
    assert len(on) == math.floor(D / cp) == 4
    r_on = D - 4 * cp
    assert len(off) == math.floor((D - r_on) / cn) == 2
    assert float(lr[0, 0]) == 4 * cp - 2 * cn


def test_event_count_cap_255():
    frames = np.array([100.0], np.float32).reshape(1, 1, 1)
    ev, lr = orc.event_frames(frames, np.zeros((1, 1), np.float32), 0.125, 0.125, 1.0)
    assert len(ev) == 255 and float(lr[0, 0]) == 255 * 0.125


# ---- P11: threshold mismatch, Eq. 8: per-pixel theta_ON / theta_OFF ------------------------
def test_p11_per_pixel_thresholds_closed_form():
    """Every pixel follows Eq. 4 with ITS OWN thresholds: an up-ramp of D then a down-ramp back to 0 gives
    floor(D / theta_on(u)) ON events and floor((D - r_on(u)) / theta_off(u)) OFF events, r_on the ON residual.
    Dyadic thresholds and endpoints keep binary32 exact; the scalar c_pos / c_neg passed alongside are absurd
    on purpose (a map that is ignored, or ON / OFF maps that are swapped, changes the counts)."""
    th_on = np.array([[0.125, 0.25, 0.5], [0.25, 0.5, 0.125]], np.float32)
    th_off = np.array([[0.5, 0.125, 0.25], [0.25, 0.25, 0.5]], np.float32)
    H, W = th_on.shape
    D = np.float32(2.1875)
    up = np.linspace(0.0, float(D), 8, dtype=np.float64)[1:]
    frames = np.concatenate([up, up[::-1][1:], [0.0]]).astype(np.float32)
    frames = np.broadcast_to(frames[:, None, None], (len(frames), H, W)).copy()
    ev, lr = orc.event_frames(frames, np.zeros((H, W), np.float32), 7.0, 9.0, 1.0, theta_on=th_on, theta_off=th_off)
    for y in range(H):
        for x in range(W):
            on = sum(1 for e in ev if e["x"] == x and e["y"] == y and e["p"] > 0)
            off = sum(1 for e in ev if e["x"] == x and e["y"] == y and e["p"] < 0)
            n_on = math.floor(float(D) / float(th_on[y, x]))
            top = n_on * float(th_on[y, x])                       # reference level after the up-ramp
            n_off = math.floor(top / float(th_off[y, x]))
            assert (on, off) == (n_on, n_off), (y, x, on, off, n_on, n_off)
            assert float(lr[y, x]) == top - n_off * float(th_off[y, x])


def test_p11b_constant_maps_equal_the_scalar_thresholds():
    """Special case that reduces to Eq. 4 with one C: maps filled with (C+, C-) give the scalar result, event
    for event (count, polarity, timestamp) and bit for bit in L_ref."""
    r = _rng(11)
    S, H, W = 12, 5, 6
    frames = np.cumsum(r.normal(0, 0.3, size=(S, H, W)), axis=0).astype(np.float32)
    L0 = np.zeros((H, W), np.float32)
    ev0, lr0 = orc.event_frames(frames, L0, 0.2, 0.3, 1.0)
    ev1, lr1 = orc.event_frames(frames, L0, 5.0, 5.0, 1.0, theta_on=np.full((H, W), 0.2, np.float32),
                                theta_off=np.full((H, W), 0.3, np.float32))
    assert len(ev0) == len(ev1) > 0 and np.array_equal(ev0, ev1) and np.array_equal(lr0, lr1)


# ---- P12: refractory period [R26] --------------------------------------------------------------
def _greedy(times, tau, t_last=-math.inf):
    out = []
    for k, t in enumerate(times, start=1):
        if t - t_last >= tau:
            out.append(k)
            t_last = t
    return out


@pytest.mark.parametrize("tau_num,expect_stride", [(2.5, 3), (3.0, 3), (3.0625, 4), (0.5, 1)])
def test_p12_refractory_on_a_linear_ramp(tau_num, expect_stride):
    """L rises by 4.0 = 32 C over one interval, sampled at S = 8 frames: the crossings fall at t_k = k / 32
    (dyadic, exact in binary32).  With tau_r = tau_num / 32 the emitted crossings are the greedy subsequence
    with gaps >= tau_r (>= : a gap of exactly tau_r is emitted), computed here on exact rationals; L_ref is the
    same as without a refractory period (it follows every crossing)."""
    C, S, T = 0.125, 8, 1.0
    frames = (np.arange(1, S + 1, dtype=np.float32) * np.float32(0.5)).reshape(S, 1, 1)
    L0 = np.zeros((1, 1), np.float32)
    tau = tau_num / 32.0
    ev, lr, tl = orc.event_frames(frames, L0, C, C, T, tau_r=tau)
    ev0, lr0 = orc.event_frames(frames, L0, C, C, T)
    assert len(ev0) == 32 and float(lr[0, 0]) == float(lr0[0, 0]) == 4.0
    want = _greedy([k / 32.0 for k in range(1, 33)], tau)
    assert want == list(range(1, 33, expect_stride))
    got = [round(float(e["t_off"]) * 32) for e in ev]
    assert got == want and all(abs(float(e["t_off"]) - k / 32.0) < 1e-7 for e, k in zip(ev, want))
    assert all(int(e["p"]) == 1 for e in ev)
    assert float(tl[0, 0]) == want[-1] / 32.0


def test_p12b_refractory_state_carries_into_the_frames():
    """t_last0 = -1/64 (an event 1/64 s before the interval started), tau_r = 3/64: the first crossing at
    t = 1/32 = 2/64 has a gap of exactly 3/64 and is emitted; with t_last0 = -1/128 it is suppressed and the
    second (t = 2/32) is the first one out."""
    C, S, T = 0.125, 8, 1.0
    frames = (np.arange(1, S + 1, dtype=np.float32) * np.float32(0.5)).reshape(S, 1, 1)
    L0 = np.zeros((1, 1), np.float32)
    for t0, first in ((-1.0 / 64, 1), (-1.0 / 128, 2)):
        ev, lr, tl = orc.event_frames(frames, L0, C, C, T, tau_r=3.0 / 64, t_last0=np.full((1, 1), t0, np.float32))
        times = [k / 32.0 for k in range(1, 33)]
        want = _greedy(times, 3.0 / 64, t0)
        assert want[0] == first
        assert [round(float(e["t_off"]) * 32) for e in ev] == want


def test_p12c_refractory_across_intervals_in_the_full_oracle():
    """Whole oracle, three intervals of a flickering uniform scene (zero motion): consecutive emitted events of a
    pixel are at least tau_r apart in absolute time, also across keyframes (t_last is carried, shifted by T);
    events are a subset of the run without refractory period with the same stamps; L_ref is unchanged."""
    E, H, W, S, T, C, tau = 1, 3, 4, 4, 1.0 / 60.0, 0.2, 0.004
    r = _rng(12)
    kfs = []
    for k in range(4):
        lum = np.exp(r.uniform(-2.0, 2.0, size=(E, H, W))).astype(np.float32)
        kfs.append(dict(rad=np.repeat(lum[..., None], 3, axis=-1).copy(), mv=np.zeros((E, H, W, 2), np.float32),
                        z=np.ones((E, H, W), np.float32)))
    o_ref = orc.Oracle(E, H, W, S, C, C, 1e-3, T, tau_r=tau)
    o_all = orc.Oracle(E, H, W, S, C, C, 1e-3, T)
    ev_ref, ev_all = [], []
    for kf in kfs:
        ev_ref.append(o_ref.step(kf["rad"], kf["mv"], kf["z"]))
        ev_all.append(o_all.step(kf["rad"], kf["mv"], kf["z"]))
    assert np.array_equal(o_ref.Lref, o_all.Lref)
    a, b = np.concatenate(ev_ref), np.concatenate(ev_all)
    assert 0 < len(a) < len(b)
    key = lambda e: (int(e["kf"]), int(e["y"]), int(e["x"]), int(e["substep"]), int(e["k"]))
    tb = {key(e): float(e["t_off"]) for e in b}
    assert all(key(e) in tb and abs(tb[key(e)] - float(e["t_off"])) < 1e-6 for e in a)
    last = {}
    for e in a:                                                   # stream order is time order per pixel
        p, t = (int(e["y"]), int(e["x"])), int(e["kf"]) * T + float(e["t_off"])
        if p in last:
            assert t - last[p] >= tau - 1e-6
        last[p] = t
    for (y, x), t in last.items():                                # carried state = last stamp relative to the NEXT interval
        assert abs(float(o_ref.t_last[0, y, x]) - (t - 3 * T)) < 1e-6


# ---- P13: over-render margin and crop (Supp. B 317-319) [R27] ------------------------------------
def test_p13_margin_removes_the_border_artifacts_of_a_translation():
    """A textured plane translating by D = S d per keyframe (integer d, S a power of two).  On the plain frame the
    strip that enters the field of view is seen by neither keyframe at some substeps (holes, held values); with a
    margin >= |D| rendered around it and cropped after the warp, the events of the cropped frame are exactly those
    of the ANALYTIC frame sequence L(t_i) fed to the event stage (which has its own pins), at the cropped
    coordinates, and no hole is left inside the crop."""
    H, W, S, dx, dy, M = 14, 18, 4, 2, -1, 8            # |D| = (8, 4) <= M
    He, We = H + 2 * M, W + 2 * M
    r = _rng(13)
    big = r.uniform(-3, 3, size=(He + 96, We + 96)).astype(np.float32)
    yse, xse = np.mgrid[0:He, 0:We]
    tex_e = lambda px, py: big[yse - py + 48, xse - px + 48]          # extended frame, surface moved by (px, py)
    crop = lambda a: a[..., M:M + H, M:M + W]
    C = 0.25

    def run(margin):
        h, w = (He, We) if margin else (H, W)
        o = orc.Oracle(1, h, w, S, C, C, 1e-3, 1.0, debug=True, margin=margin)
        mv = np.empty((1, h, w, 2), np.float32)
        mv[..., 0], mv[..., 1] = -S * dx, -S * dy
        depth = np.full((1, h, w), 3.0, np.float32)
        evs = []
        for k in range(3):
            L = tex_e(k * S * dx, k * S * dy)
            L = L if margin else crop(L)
            evs.append(o.step(_rad_from_L(L)[None], mv, depth))
        return o, np.concatenate(evs)

    o_m, ev_m = run(M)
    o_0, ev_0 = run(0)
    assert o_m.holes == 0 and o_0.holes > 0
    # analytic sequence of the cropped frame: keyframes through the oracle's own log (same rounding), substeps exact
    L0 = orc.log_luminance(_rad_from_L(tex_e(0, 0))[None], 1e-3)[0]
    Lk = lambda k, i: crop(orc.log_luminance(_rad_from_L(tex_e((k * S + i) * dx, (k * S + i) * dy))[None], 1e-3)[0])
    lref, lprev, want = crop(L0).copy(), crop(L0).copy(), []
    for k in range(2):
        frames = np.stack([Lk(k, i) for i in range(1, S + 1)])
        e, lref = orc.event_frames(frames, lprev, C, C, 1.0, Lref0=lref)
        lprev = frames[-1]
        want += [(k, int(v["substep"]), int(v["y"]), int(v["x"]), int(v["p"])) for v in e]
    got = [(int(v["kf"]), int(v["substep"]), int(v["y"]), int(v["x"]), int(v["p"])) for v in ev_m]
    assert sorted(got) == sorted(want) and len(got) > 0
    assert all(0 <= y < H and 0 <= x < W for (_, _, y, x, _) in got)
    got0 = [(int(v["kf"]), int(v["substep"]), int(v["y"]), int(v["x"]), int(v["p"])) for v in ev_0]
    assert sorted(got0) != sorted(want)                     # the plain frame does show the border artifact


# ---- P14: colour events [R28] ---------------------------------------------------------------------
def test_p14_channel_log_is_the_log_of_that_channel_alone():
    """"Replacing I with individual R, G, B channels": L = log(channel + eps) by math.log in double, rounded once
    to binary32; the other two channels do not matter (they hold absurd values), negative values clamp to 0."""
    r = _rng(14)
    n, eps = 200, 1e-3
    for ch in (0, 1, 2):
        rad = r.uniform(-1e6, 1e6, size=(n, 3)).astype(np.float32)
        rad[:, ch] = np.exp(r.uniform(-7, 7, size=n)).astype(np.float32)
        rad[:5, ch] = [-1.0, 0.0, 1e-30, 1.0, 1e6]
        L = orc.log_luminance(rad, eps, channel=ch)
        for i in range(n):
            c = max(float(rad[i, ch]), 0.0)
            assert L[i] == np.float32(math.log(c + float(np.float32(eps))))
    # a grey pixel has the same log in every channel, and its luminance log is within rounding of it
    g = np.full((1, 3), 0.37, np.float32)
    Ls = [float(orc.log_luminance(g, eps, channel=c)[0]) for c in (0, 1, 2)]
    assert Ls[0] == Ls[1] == Ls[2] and abs(Ls[0] - float(orc.log_luminance(g, eps)[0])) < 1e-6


def test_p14b_colour_events_are_three_independent_runs():
    """A scene whose RED channel alone changes between keyframes: the R run fires, the G and B runs stay silent,
    and the R run equals the luminance run of the grey image made of that channel (same warp, same Eq. 4)."""
    E, H, W, S, T, C = 1, 4, 5, 4, 1.0 / 60.0, 0.2
    r = _rng(15)
    base = np.exp(r.uniform(-1, 1, size=(E, H, W, 3))).astype(np.float32)
    nxt = base.copy()
    nxt[..., 0] *= np.float32(3.0)
    mv, z = np.zeros((E, H, W, 2), np.float32), np.ones((E, H, W), np.float32)
    n_ev = []
    for ch in (0, 1, 2):
        o = orc.Oracle(E, H, W, S, C, C, 1e-3, T, channel=ch)
        o.step(base, mv, z)
        n_ev.append(len(o.step(nxt, mv, z)))
    assert n_ev[0] == H * W * math.floor(math.log(3.0) / C) and n_ev[1] == n_ev[2] == 0


# ---- P15: noise events (Eq. 9-10) [R29] --------------------------------------------------------
def test_p15_generator_is_splitmix64_and_its_fields_are_uniform():
    """The counter hash is the published splitmix64 output function: with key + 4 i + s equal to the golden-ratio
    increment it must return the first output of splitmix64 seeded with 0 (known test vector).  Its 24-bit fields
    are uniform and the three streams are uncorrelated."""
    L = orc.lib()
    G = 0x9E3779B97F4A7C15
    assert L.evo_noise_hash((G - 4) & (2 ** 64 - 1), 1, 0) == 0xE220A8397B1DCDAF
    assert L.evo_noise_hash((2 * G - 6) & (2 ** 64 - 1), 1, 2) == 0x6E789E6AA1B965F4
    key = [L.evo_noise_key(12345, 3, 1, q) for q in range(4000)]
    assert len(set(key)) == 4000
    f = lambda h, sh: ((h >> sh) & 0xFFFFFF) / 2.0 ** 24
    u = np.array([[f(L.evo_noise_hash(k, i, s), sh) for s in (0, 1, 2) for sh in (40, 16)] for k in key for i in (1, 2, 3)])
    assert np.all(np.abs(u.mean(axis=0) - 0.5) < 4 * (1 / 12 / len(u)) ** 0.5)
    hist = np.stack([np.histogram(u[:, c], bins=16, range=(0, 1))[0] for c in range(u.shape[1])])
    chi2 = ((hist - len(u) / 16) ** 2 / (len(u) / 16)).sum(axis=1)
    assert np.all(chi2 < 45.0)                                   # 15 dof: P(chi2 > 45) ~ 8e-5
    cc = np.corrcoef(u.T)
    assert np.all(np.abs(cc - np.eye(u.shape[1])) < 0.04)


def test_p15b_exp32_is_exp():
    xs = np.concatenate([np.linspace(-20, 20, 4001), [-79.9, 79.9, 0.0, -0.0, 1e-8]]).astype(np.float32)
    for x in xs:
        got, want = orc.lib().evo_exp32(float(x)), math.exp(float(x))
        assert abs(got - want) <= 6e-7 * want, (x, got, want)
    assert orc.lib().evo_exp32(-1000.0) == 0.0 and orc.lib().evo_exp32(float("nan")) == 0.0
    assert orc.lib().evo_exp32(1000.0) == orc.lib().evo_exp32(80.0)


def _noise_run(L_value, noise, S=64, H=40, W=50, T=1.0):
    frames = np.full((S, H, W), L_value, np.float32)
    ev, lr = orc.event_frames(frames, frames[0], 0.2, 0.2, T, noise=noise)
    return ev, S * H * W, T / S


def test_p15c_leak_rate_polarity_and_stamps():
    """Static scene, leak only: every pixel-substep is a Bernoulli trial with P = r_l dt (Eq. 9); the events are ON,
    their stamps uniform inside their substep; another seed gives another draw; zero rates give nothing."""
    noise = dict(seed=7, r_leak=3.2, eps=1e-3)
    ev, N, dt = _noise_run(0.0, noise)
    P = 3.2 * dt
    assert abs(len(ev) - N * P) < 4 * (N * P * (1 - P)) ** 0.5
    assert np.all(ev["p"] == 1) and np.all(ev["k"] == 1001)
    fr = ev["t_off"] / dt - (ev["substep"] - 1)
    assert np.all((fr >= 0) & (fr < 1)) and abs(fr.mean() - 0.5) < 4 * (1 / 12 / len(ev)) ** 0.5
    ev2, _, _ = _noise_run(0.0, dict(noise, seed=8))
    assert len(ev2) != len(ev) or not np.array_equal(ev2["x"], ev["x"])
    assert len(_noise_run(0.0, dict(seed=7, eps=1e-3))[0]) == 0


def test_p15d_shot_rate_falls_with_intensity():
    """Eq. 10: P_shot = r_s dt (1 - Ibar).  Black (I = 0): the full rate; I = I_white / 2: half of it; I >= I_white:
    none.  Polarity is a fair coin."""
    eps, iw = 1e-3, 2.0
    for I, frac in ((0.0, 1.0), (1.0, 0.5), (2.0, 0.0), (50.0, 0.0)):
        ev, N, dt = _noise_run(math.log(I + eps), dict(seed=11, r_shot=6.4, i_white=iw, eps=eps))
        P = 6.4 * dt * frac
        assert abs(len(ev) - N * P) <= 4 * (N * P * (1 - P)) ** 0.5 + (0 if frac else 0), (I, len(ev), N * P)
        if frac:
            assert np.all(ev["k"] == 1002) and abs((ev["p"] == 1).mean() - 0.5) < 4 * 0.5 / len(ev) ** 0.5


def test_p15e_hot_pixels_and_signal_untouched():
    """Hot pixels fire only inside H, at r_h dt; with all three sources on, the threshold crossings, their stamps
    and L_ref are those of the noise-free run (noise events leave L_ref alone)."""
    S, H, W = 64, 40, 50
    hot = np.zeros((H, W), np.uint8)
    hot[::5, ::7] = 1
    ev, N, dt = _noise_run(0.0, dict(seed=3, r_hot=16.0, eps=1e-3, hot=hot), S, H, W)
    n_hot = int(hot.sum()) * S
    P = 16.0 * dt
    assert np.all(hot[ev["y"], ev["x"]] == 1) and np.all(ev["k"] == 1003)
    assert abs(len(ev) - n_hot * P) < 4 * (n_hot * P * (1 - P)) ** 0.5
    r = _rng(16)
    frames = np.cumsum(r.normal(0, 0.15, size=(S, H, W)), axis=0).astype(np.float32)
    L0 = np.zeros((H, W), np.float32)
    a, lra = orc.event_frames(frames, L0, 0.2, 0.3, 1.0)
    b, lrb = orc.event_frames(frames, L0, 0.2, 0.3, 1.0, noise=dict(seed=3, r_leak=2.0, r_shot=2.0, r_hot=9.0, eps=1e-3, hot=hot))
    sig = b[b["k"] < 1000]
    assert np.array_equal(lra, lrb) and len(b) > len(a) and np.array_equal(sig, a)


# ------------------------------------------------------------------------------------------------
# P19: defocus (reading R31): separable Gaussian on the warped LINEAR frame, then the log
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sigma", [0.1, 0.3, 0.5, 1.0, 2.3])
def test_p19_defocus_kernel_is_the_library_gaussian_filter(sigma):
    """Taps: R = ceil(3 sigma), symmetric, sum 1; the two-pass blur equals scipy.ndimage.gaussian_filter (truncated at
    the same radius, replicated border) and the 2-D correlation with the outer product of the taps (separability)."""
    from scipy import ndimage
    w = orc.gauss_taps(sigma)
    R = (w.size - 1) // 2
    assert R == math.ceil(3 * sigma) and np.array_equal(w, w[::-1]) and abs(float(w.astype(np.float64).sum()) - 1) < 1e-6
    assert abs(w[R + 1] / w[R] - math.exp(-1 / (2 * sigma * sigma))) < 1e-6 * max(1.0, w[R + 1] / w[R])
    f = _rng(19).uniform(0.0, 7.0, (23, 31)).astype(np.float32)
    got = orc.blur(f, w).astype(np.float64)
    lib_ = ndimage.gaussian_filter(f.astype(np.float64), sigma, mode="nearest", radius=R)
    assert np.abs(got - lib_).max() < 3e-6
    two_d = ndimage.correlate(f.astype(np.float64), np.outer(w, w).astype(np.float64), mode="nearest")
    assert np.abs(got - two_d).max() < 3e-6
    const = np.full((9, 11), 3.25, np.float32)
    assert np.abs(orc.blur(const, w) - 3.25).max() < 1e-6 * 3.25 * (2 * R + 2)


def test_p19b_defocus_blurs_the_linear_frame_with_holes_held_unblurred():
    """The frame the event model sees = log(blur(warped LINEAR frame) + eps), a hole holding its previous UNBLURRED
    value: rebuilt here from the plain run's winners (pinned by P3 / P4 / P5), numpy's luminance, scipy's filter and
    np.log.  The alternatives (blur of the log frame; holes holding the blurred value) miss by far more than the
    tolerance on this scene, so the pin tells them apart."""
    from scipy import ndimage
    H, W, S, dx, dy, sigma, eps = 20, 26, 4, 2, -1, 0.8, 1e-3
    r = _rng(23)
    big = r.uniform(-3, 3, size=(H + 64, W + 64)).astype(np.float32)
    ys, xs = np.mgrid[0:H, 0:W]
    tex = lambda px, py: big[ys - py + 32, xs - px + 32]
    mv = np.empty((1, H, W, 2), np.float32)
    mv[..., 0], mv[..., 1] = -S * dx, -S * dy
    depth = np.full((1, H, W), 3.0, np.float32)
    rads = [_rad_from_L(tex(0, 0))[None], _rad_from_L(tex(S * dx, S * dy))[None], _rad_from_L(tex(2 * S * dx, 2 * S * dy))[None]]
    plain = orc.Oracle(1, H, W, S, 0.2, 0.2, eps, 1 / 60, debug=True)
    blur_ = orc.Oracle(1, H, W, S, 0.2, 0.2, eps, 1 / 60, debug=True, defocus_sigma=sigma)
    lin = lambda rad: ((0.2126 * rad[..., 0].astype(np.float64) + 0.7152 * rad[..., 1]) + 0.0722 * rad[..., 2]).clip(0).astype(np.float32)
    w = orc.gauss_taps(sigma)
    R = (w.size - 1) // 2
    filt = lambda f: ndimage.gaussian_filter(f.astype(np.float64), sigma, mode="nearest", radius=R)
    e32 = np.float64(np.float32(eps))
    held = lin(rads[0])[0]                               # the unblurred warped frame carried through the holes
    held_alt = filt(held)                                # alternative: holes hold the BLURRED value
    n_holes, worst_alt1, worst_alt2 = 0, 0.0, 0.0
    for k, rad in enumerate(rads):
        plain.step(rad, mv, depth)
        ev = blur_.step(rad, mv, depth)
        if k == 0:
            L0 = np.log(filt(lin(rad)[0]) + e32)
            assert np.abs(blur_.Lref[0] - L0).max() < 3e-6 and len(ev) == 0
            continue
        IA, IB = lin(rads[k - 1])[0].ravel(), lin(rad)[0].ravel()
        for i in range(S):
            d, idx = plain.dbg["dir"][0, i], plain.dbg["idx"][0, i].astype(np.int64)
            assert np.array_equal(d, blur_.dbg["dir"][0, i]) and np.array_equal(idx, blur_.dbg["idx"][0, i].astype(np.int64))
            safe = np.where(d == 3, 0, idx)
            frame = np.where(d == 0, IB[safe], np.where(d == 1, IA[safe], held))
            frame_alt = np.where(d == 0, IB[safe], np.where(d == 1, IA[safe], held_alt))
            n_holes += int((d == 3).sum())
            want = np.log(filt(frame) + e32)
            got = blur_.dbg["Lhat"][0, i].astype(np.float64)
            assert np.abs(got - want).max() < 5e-6, (k, i, float(np.abs(got - want).max()))
            worst_alt1 = max(worst_alt1, float(np.abs(got - filt(np.log(frame.astype(np.float64) + e32))).max()))
            worst_alt2 = max(worst_alt2, float(np.abs(got - np.log(filt(frame_alt) + e32)).max()))
            held, held_alt = frame, filt(frame_alt)
    assert n_holes > 0 and worst_alt1 > 1e-2 and worst_alt2 > 1e-3


def test_p19c_zero_sigma_is_the_plain_run():
    """sigma = 0 (one tap of weight 1): the frames are the plain frames up to the rounding of the linear intensity to
    binary32 before the log, and the events are the plain events."""
    spec = scenes.small(scenes.config(1), height=40, width=56, num_keyframes=3)
    sc = scenes.make_scene(spec)
    a = orc.Oracle(1, spec.height, spec.width, spec.substeps, spec.c_pos, spec.c_neg, spec.log_eps, spec.keyframe_dt, debug=True)
    b = orc.Oracle(1, spec.height, spec.width, spec.substeps, spec.c_pos, spec.c_neg, spec.log_eps, spec.keyframe_dt, debug=True,
                   defocus_sigma=0.0)
    na = nb = 0
    for k in range(3):
        kf = {key: v.numpy() for key, v in scenes.render_keyframe(sc, k).items()}
        ea = a.step(kf["rad"], kf["mv_bwd"], kf["depth"], kf["mv_fwd"])
        eb = b.step(kf["rad"], kf["mv_bwd"], kf["depth"], kf["mv_fwd"])
        na, nb = na + len(ea), nb + len(eb)
        if k:
            assert np.abs(a.dbg["Lhat"].astype(np.float64) - b.dbg["Lhat"]).max() < 1e-6
    assert na > 100 and abs(na - nb) <= max(2, na // 500)          # rounding of I before the log moves a few ties


def test_p19d_defocus_softens_edges_and_a_static_scene_stays_silent():
    """A static scene fires nothing with defocus on (the blurred frame is constant in time); on the moving scene the
    blur lowers the largest log step between neighbouring pixels."""
    spec = scenes.small(scenes.config(1), height=40, width=56, num_keyframes=3)
    sc = scenes.make_scene(spec)
    kf = {key: v.numpy() for key, v in scenes.render_keyframe(sc, 0).items()}
    o = orc.Oracle(1, spec.height, spec.width, spec.substeps, spec.c_pos, spec.c_neg, spec.log_eps, spec.keyframe_dt,
                   defocus_sigma=0.5)
    zero = np.zeros_like(kf["mv_bwd"])
    assert len(o.step(kf["rad"], zero, kf["depth"])) == 0
    assert len(o.step(kf["rad"], zero, kf["depth"])) == 0 and o.holes == 0
    sharp = orc.log_luminance(kf["rad"], spec.log_eps)[0]
    soft = o.Lprev[0]
    assert np.abs(np.diff(soft, axis=1)).max() < np.abs(np.diff(sharp, axis=1)).max()


# ------------------------------------------------------------------------------------------------
# P20: weighted front-surface splat (reading R32; composite mode 2)
# ------------------------------------------------------------------------------------------------
def _brute_weighted(H, W, i, S, src_is_B, disp, Zsrc, Zoth, Lsrc):
    """Gather form straight from the definition: per target, the sources covering it with positive bilinear weight,
    the nearest depth Z*, the front set zt <= 1.01 Z*, the weighted mean of their log values -- in exact float64
    (dyadic inputs).  Returns (mean [H,W] float64 with NaN where nothing lands, spread of L among the contributors)."""
    f = i / S
    wgt = (1 - f) if src_is_B else f
    out = np.full((H, W), np.nan)
    spread = np.zeros((H, W))
    for ty in range(H):
        for tx in range(W):
            c = []
            for sy in range(H):
                for sx in range(W):
                    dx, dy = float(disp[sy, sx, 0]), float(disp[sy, sx, 1])
                    qx, qy = sx + wgt * dx, sy + wgt * dy
                    if not (abs(qx - tx) < 1 and abs(qy - ty) < 1):
                        continue
                    jx, jy = math.floor(sx + dx + 0.5), math.floor(sy + dy + 0.5)
                    zs = float(Zsrc[sy, sx])
                    zo = float(Zoth[jy, jx]) if (0 <= jx < W and 0 <= jy < H) else zs
                    za, zb = (zo, zs) if src_is_B else (zs, zo)
                    c.append(((1 - f) * za + f * zb, (1 - abs(qx - tx)) * (1 - abs(qy - ty)), float(Lsrc[sy, sx])))
            if c:
                zmin = min(z for z, _, _ in c)
                front = [(w_, l_) for z, w_, l_ in c if z <= float(np.float32(1.01)) * zmin]
                out[ty, tx] = sum(w_ * l_ for w_, l_ in front) / sum(w_ for w_, _ in front)
                spread[ty, tx] = max(l_ for _, l_ in front) - min(l_ for _, l_ in front)
    return out, spread


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_p20_weighted_splat_is_the_front_surface_mean_8x8(seed):
    """The oracle's integer sums (weights in units of 2^-20, at least one; log values in units of 2^-24) against the exact
    float64 gather form: within the quantisation bound 2^-19 x (spread of the contributors' L) + 2^-23."""
    H = W = 8
    S = 4
    r = _rng(200 + seed)
    levels = np.array([1.0, 1.005, 1.5, 2.0, 3.0], np.float32)     # 1.0 / 1.005: inside the 1 % band; the rest outside
    n_multi = 0
    for src_is_B in (True, False):
        disp = (r.integers(-12, 13, size=(H, W, 2)) / 4.0).astype(np.float32)
        Zsrc = levels[r.integers(0, len(levels), size=(H, W))]
        Zoth = Zsrc.copy()                                           # both ends alike: zt = the source's level, exactly
        Lsrc = (r.integers(-40, 41, size=(H, W)) / 8.0).astype(np.float32)
        for i in range(1, S + 1):
            z = orc.splat(i, S, src_is_B, disp, Zsrc, Zoth)
            acc = orc.wsplat(i, S, src_is_B, disp, Zsrc, Zoth, Lsrc, z)
            want, spread = _brute_weighted(H, W, i, S, src_is_B, disp, Zsrc, Zoth, Lsrc)
            hit = z != EMPTY
            assert np.array_equal(hit, ~np.isnan(want)) and np.all(acc[..., 1][hit] > 0) and not acc[~hit].any()
            got = acc[..., 0][hit] / acc[..., 1][hit] / 2.0 ** 24
            assert np.all(np.abs(got - want[hit]) <= 2.0 ** -19 * spread[hit] + 2.0 ** -23), (seed, src_is_B, i)
            n_multi += int((spread[hit] > 0).sum())
    assert n_multi > 50                                             # the mean really mixes different values


def test_p20b_weighted_splat_closed_forms():
    """(a) Integer translation: every weight is 0 or 1, the weighted mode IS the winner-take-all mode, frames and events.
    (b) A half-pixel shift of a fronto-parallel plane: every target is the mean of its two neighbours' log values.
    (c) A near square over a far plane: the far sources under it are behind the front surface and carry no weight; a
    source within 1 % of the front depth does."""
    H, W, S = 12, 16, 4
    r = _rng(31)
    L0 = (r.integers(-24, 25, size=(H, W)) / 8.0).astype(np.float32)
    depth = np.full((H, W), 4.0, np.float32)
    # (a)
    mv = np.zeros((1, H, W, 2), np.float32); mv[..., 0] = -S * 1.0
    big = r.uniform(-2, 2, size=(H + 64, W + 64)).astype(np.float32)
    ys, xs = np.mgrid[0:H, 0:W]
    tex = lambda px: big[ys + 32, xs - px + 32]
    frames = {}
    for mode in (0, 2):
        o = orc.Oracle(1, H, W, S, 0.2, 0.2, 1e-3, 1 / 60, composite_mode=mode, debug=True)
        o.step(_rad_from_L(tex(0))[None], mv, depth[None])
        ev = o.step(_rad_from_L(tex(S))[None], mv, depth[None])
        frames[mode] = (o.dbg["Lhat"].copy(), o.dbg["dir"].copy(), len(ev))
    assert np.array_equal(frames[0][1], frames[2][1]) and frames[0][2] == frames[2][2] > 0
    assert np.abs(frames[0][0].astype(np.float64) - frames[2][0]).max() <= 2.0 ** -24      # only the 2^-24 grid of L
    # (b)
    disp = np.zeros((H, W, 2), np.float32); disp[..., 0] = 2.0       # at i = 1 of S = 4 the shift is (1 - f) 2 = 1.5 px
    z = orc.splat(1, S, True, disp, depth, depth)
    acc = orc.wsplat(1, S, True, disp, depth, depth, L0, z)
    got = acc[..., 0] / np.maximum(acc[..., 1], 1) / 2.0 ** 24
    want = (L0[:, 1:-2].astype(np.float64) + L0[:, 2:-1]) / 2        # target x >= 3: sources x - 2 and x - 1, half a weight each
    assert np.array_equal(acc[:, 3:, 1], np.full((H, W - 3), 2 ** 20))  # two half weights
    assert np.abs(got[:, 3:] - want).max() < 2.0 ** -23
    # (c)
    Z = np.full((H, W), 8.0, np.float32); Z[4:8, 5:9] = 2.0; Z[4, 5] = 2.01                # 2.01 <= 1.01 * 2.0
    disp = np.full((H, W, 2), 0.5, np.float32)                      # everything moves by (1 - f) 0.5: fractional weights
    Lc = np.where(Z > 3, 5.0, -3.0).astype(np.float32); Lc[4, 5] = -1.0
    z = orc.splat(2, S, True, disp, Z, Z)
    acc = orc.wsplat(2, S, True, disp, Z, Z, Lc, z)
    got = acc[..., 0] / np.maximum(acc[..., 1], 1) / 2.0 ** 24
    inside = got[5:8, 6:9]                                           # fully under the square: only near sources count
    assert np.all(inside < -0.9) and np.all(np.abs(got[9:, 10:] - 5.0) < 1e-6)
    assert -3.0 < got[5, 6] < -2.0                                   # the 2.01-deep source (L = -1) is mixed in with the -3s
