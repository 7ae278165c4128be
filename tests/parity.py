"""Shared machinery of the GPU parity tests: run the CUDA library (through the C ABI) and the CPU
oracle on the same seeded keyframes and compare them the way north_star prescribes:

* composite winner (direction, source index) per pixel-substep: bit-exact;
* warped log-luminance: within 1e-5 absolute;
* events as multisets of (env, x, y, substep, polarity): bit-exact, except at threshold ties where
  ||dL| - k C| < 1e-5 for an integer k (R5) -- the number of ties is returned and reported;
* timestamps: within 1e-7 s;
* carried state L_ref, L_prev.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence

import numpy as np
import torch

from oracle import evis_oracle as orc
from paper_2607_08098_b200 import binding, scenes

TOL_L = 1e-5
TOL_T = 1e-7
TOL_TIE = 1e-5


@dataclass
class ParityReport:
    steps: int = 0
    events_gpu: int = 0
    events_oracle: int = 0
    ties: int = 0
    winner_mismatch: int = 0
    max_dL: float = 0.0
    max_dt: float = 0.0
    holes: int = 0
    notes: List[str] = field(default_factory=list)


def canon_gpu(ev: np.ndarray) -> np.ndarray:
    """Sort library events into the canonical comparison order (env, substep, y, x, t)."""
    order = np.lexsort((ev["t_off"], ev["x"], ev["y"], ev["substep"], ev["env"]))
    return ev[order]


def canon_oracle(ev: np.ndarray) -> np.ndarray:
    order = np.lexsort((ev["k"], ev["x"], ev["y"], ev["substep"], ev["env"]))
    return ev[order]


def _counts(ev, E, S, H, W, env_map=None):
    """Signed event count per (env, substep, y, x): +n for ON, -n for OFF (one polarity per cell)."""
    c = np.zeros((E, S, H, W), np.int32)
    env = ev["env"].astype(np.int64)
    if env_map is not None:
        env = env_map[env]
    np.add.at(c, (env, ev["substep"].astype(np.int64) - 1, ev["y"].astype(np.int64), ev["x"].astype(np.int64)),
              ev["p"].astype(np.int32))
    return c


def compare_step(gpu_ev: np.ndarray, ora_ev: np.ndarray, ora: orc.Oracle, E: int, S: int, H: int, W: int,
                 c_pos: float, c_neg: float, rep: ParityReport, kf: int,
                 gpu_dbg=None, env_sel: Optional[Sequence[int]] = None, thresholds=None, margin: int = 0) -> None:
    """Compare one step.  ``env_sel``: the oracle ran only these envs of the GPU batch (oracle env j =
    GPU env env_sel[j]); GPU events of other envs are ignored."""
    if env_sel is not None:
        env_map = np.full(65536, -1, np.int64)
        env_map[np.asarray(env_sel)] = np.arange(len(env_sel))
        keep = env_map[gpu_ev["env"].astype(np.int64)] >= 0
        gpu_ev = gpu_ev[keep].copy()
        gpu_ev["env"] = env_map[gpu_ev["env"].astype(np.int64)].astype(np.uint16)
    Eo = E if env_sel is None else len(env_sel)
    M = margin                                     # H, W: the over-rendered frame; events live in the crop (R27)
    Hc, Wc = H - 2 * M, W - 2 * M
    inner = (Ellipsis, slice(M, H - M), slice(M, W - M))
    assert np.all(gpu_ev["kf"] == kf)
    rep.steps += 1
    rep.events_gpu += len(gpu_ev)
    rep.events_oracle += len(ora_ev)

    # --- warp parity through the debug hook ---------------------------------------------------
    if gpu_dbg is not None:
        win, d, lh = gpu_dbg                       # [S,E,H,W]
        if env_sel is not None:
            win, d, lh = win[:, env_sel], d[:, env_sel], lh[:, env_sel]
        o_dir = np.transpose(ora.dbg["dir"], (1, 0, 2, 3))[inner]
        o_idx = np.transpose(ora.dbg["idx"], (1, 0, 2, 3))[inner]
        o_lh = np.transpose(ora.dbg["Lhat"], (1, 0, 2, 3))[inner]
        win, d, lh = win[inner], d[inner], lh[inner]
        bad = (d != o_dir) | (win != o_idx)
        rep.winner_mismatch += int(bad.sum())
        fin = np.isfinite(o_lh)                    # non-finite L (infinite radiance) must agree as such
        assert np.array_equal(fin, np.isfinite(lh)) and np.array_equal(lh[~fin], o_lh[~fin], equal_nan=True)
        if fin.any():
            rep.max_dL = max(rep.max_dL, float(np.max(np.abs(lh[fin].astype(np.float64) - o_lh[fin]))))
        rep.holes += int((o_dir == 3).sum())

    # --- events: multiset per (env, substep, y, x, polarity) -----------------------------------
    cg = _counts(gpu_ev, Eo, S, Hc, Wc)
    co = _counts(ora_ev, Eo, S, Hc, Wc)
    diff = np.argwhere(cg != co)
    if len(diff):
        # a disagreement is legitimate only at a threshold tie (R5): ||dL| - k C| < 1e-5.  It may
        # shift later counts of the same pixel, so only the FIRST disagreement of a pixel is tested.
        assert ora.dbg, "tie analysis needs the oracle's debug capture"
        seen = set()
        for e, s, y, x in diff:
            if (e, y, x) in seen:
                continue
            seen.add((e, y, x))
            dL = float(ora.dbg["dL"][e, s, y + M, x + M])
            C = c_pos if dL > 0 else c_neg
            if thresholds is not None:              # Eq. 8: the pixel's own thresholds, [Eo,H,W] numpy
                C = float((thresholds[0] if dL > 0 else thresholds[1])[e, y + M, x + M])
            k = round(abs(dL) / C)
            assert abs(abs(dL) - k * C) < TOL_TIE, \
                f"event mismatch not at a tie: env {e} substep {s + 1} ({x},{y}) dL={dL} gpu={cg[e, s, y, x]} oracle={co[e, s, y, x]}"
            rep.ties += 1
        return                                      # timestamps of this step are not comparable 1:1
    # --- timestamps ---------------------------------------------------------------------------------
    g, o = canon_gpu(gpu_ev), canon_oracle(ora_ev)
    assert len(g) == len(o)
    if len(g):
        assert np.array_equal(g["x"], o["x"]) and np.array_equal(g["y"], o["y"])
        assert np.array_equal(g["substep"].astype(np.int32), o["substep"])
        assert np.array_equal(g["p"].astype(np.int32), o["p"])
        dt = np.abs(g["t_off"].astype(np.float64) - o["t_off"])
        rep.max_dt = max(rep.max_dt, float(dt.max()))


def run_parity(spec: scenes.SceneSpec, n_keyframes: int, *, envs: Optional[Sequence[int]] = None,
               mode: int = 0, path: int = binding.PATH_GLOBAL, use_fwd: bool = True, debug: bool = True,
               capacity: int = 1 << 24, max_motion: Optional[float] = None, thresholds=None,
               tau_r: float = 0.0, margin: int = 0, channel: Optional[int] = None, mutate=None,
               render_device: str = "cuda", defocus: Optional[float] = None) -> ParityReport:
    """GPU runs the whole batch; the oracle runs ``envs`` (default: all).  Returns the report after
    asserting every bit-exact criterion; tolerances are asserted by the caller on the report."""
    sc = scenes.make_scene(spec)
    E, H, W, S = spec.num_envs, spec.height, spec.width, spec.substeps
    sel = list(range(E)) if envs is None else list(envs)
    mm = spec.max_motion_px() if max_motion is None else max_motion
    ev = binding.Evis(E, H, W, S, spec.c_pos, spec.c_neg, spec.log_eps, spec.keyframe_dt, max_motion_px=mm,
                      composite_mode=mode, path=path, event_capacity=capacity, debug_capture=debug)
    th_np = None
    if thresholds is not None:                      # (theta_on, theta_off) CUDA tensors [E,H,W] (Eq. 8)
        ev.set_thresholds(thresholds[0], thresholds[1])
        th_np = (thresholds[0][sel].cpu().numpy(), thresholds[1][sel].cpu().numpy())
    if tau_r > 0.0:                                 # refractory period
        ev.set_refractory(tau_r)
    if channel is not None:                         # colour events
        ev.set_channel(channel)
    if margin:                                      # over-render margin: spec = the over-rendered frame
        ev.set_margin(margin)
    if defocus is not None:                         # defocus
        ev.set_defocus(defocus)
    inner = (Ellipsis, slice(margin, H - margin), slice(margin, W - margin))
    ora = orc.Oracle(len(sel), H, W, S, spec.c_pos, spec.c_neg, spec.log_eps, spec.keyframe_dt,
                     composite_mode=mode, debug=True, theta_on=None if th_np is None else th_np[0],
                     theta_off=None if th_np is None else th_np[1], tau_r=tau_r, margin=margin, channel=channel,
                     defocus_sigma=defocus)
    rep = ParityReport()
    try:
        for k in range(n_keyframes):
            kf = scenes.render_keyframe(sc, k, device=render_device)
            if render_device != "cuda":             # rendered on the host (the generator is device-independent), copied over
                kf = {key: v.cuda() for key, v in kf.items()}
            if mutate is not None:                  # degenerate-input cases: the test edits the keyframe in place
                mutate(k, kf)
            fwd = kf["mv_fwd"] if use_fwd else None
            n = ev.step(kf["rad"], kf["mv_bwd"], kf["depth"], mv_fwd=fwd, sync=True)
            h = {key: v[sel].cpu().numpy() for key, v in kf.items()}
            oe = ora.step(h["rad"], h["mv_bwd"], h["depth"], h["mv_fwd"] if use_fwd else None)
            if k == 0:
                assert n == 0 and len(oe) == 0
                continue
            ge = ev.read_events()
            assert len(ge) == n
            dbg = ev.debug_read() if debug else None
            compare_step(ge, oe, ora, E, S, H, W, spec.c_pos, spec.c_neg, rep, k - 1, dbg,
                         None if envs is None else sel, th_np, margin)
            lref, lprev = ev.get_state()
            if rep.ties == 0:
                assert np.array_equal(lref[sel][inner], ora.Lref[inner]), "carried L_ref differs"
            assert np.allclose(lprev[sel][inner], ora.Lprev[inner], atol=TOL_L, rtol=0)
            if tau_r > 0.0 and rep.ties == 0:       # the carried refractory state, bit for bit (R26)
                assert np.array_equal(ev.get_t_last()[sel][inner], ora.t_last[inner]), "carried t_last differs"
            info = ev.info()
            if envs is None:
                assert info.last_holes == ora.holes
    finally:
        ev.destroy()
    assert rep.winner_mismatch == 0, f"{rep.winner_mismatch} composite winners differ"
    return rep
