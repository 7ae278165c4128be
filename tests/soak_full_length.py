"""Full-length parity soak (not collected by pytest: ~5 minutes on a B200 + one host core):

    python -m tests.soak_full_length

BASELINE.json configs 2, 3 and 4 at FULL resolution and FULL length (61 / 31 keyframes) on a few envs, the library
against the oracle step after step: events as multisets per (env, substep, pixel, polarity), timestamps, carried L_ref /
L_prev -- also in composite mode 2 (weighted splat) and with defocus.  Last run (round 2, B200): 79 398 241, 61 509 753,
68 237 477, 47 242 913 and 49 574 678 events identical, 0 ties, max |dt| 2.7e-9 s.
"""
from paper_2607_08098_b200 import scenes
from tests import parity


def main():
    for cfg, envs, kw in ((4, 5, {}), (2, 2, {}), (3, 2, {}), (4, 3, {"mode": 2}), (4, 3, {"defocus": 0.3})):
        spec = scenes.config(cfg)
        n = spec.num_keyframes
        rep = parity.run_parity(scenes.small(spec, num_envs=envs), n, debug=False, capacity=1 << 25, **kw)
        assert rep.events_gpu == rep.events_oracle and rep.max_dt <= parity.TOL_T
        print(f"cfg {cfg}, {envs} envs, {kw or 'mode 0'}: {n} keyframes, {rep.events_gpu} events identical, "
              f"ties {rep.ties}, max|dt| {rep.max_dt:.2g} s", flush=True)


if __name__ == "__main__":
    main()
