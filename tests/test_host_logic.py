"""Host-side logic that needs no GPU: the 8-byte event format of include/evis.h and the bench's readers of the committed
ncu captures."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def test_event8_layout_follows_the_header():
    """bits 0-11 x | 12-23 y | 24-39 env | 40-47 substep | 48-62 frac | 63 polarity, written out here from include/evis.h;
    decode_events8 must invert it and place the stamp at the centre of its 2^-15 cell."""
    from paper_2607_08098_b200 import binding
    rng = np.random.default_rng(3)
    n, T, S = 1000, 1.0 / 60.0, 16
    x, y = rng.integers(0, 4096, n), rng.integers(0, 4096, n)
    env, sub = rng.integers(0, 65536, n), rng.integers(1, S + 1, n)
    frac, on = rng.integers(0, 32768, n), rng.integers(0, 2, n)
    word = (x.astype(np.uint64) | (y.astype(np.uint64) << np.uint64(12)) | (env.astype(np.uint64) << np.uint64(24))
            | (sub.astype(np.uint64) << np.uint64(40)) | (frac.astype(np.uint64) << np.uint64(48))
            | (on.astype(np.uint64) << np.uint64(63)))
    ev = binding.decode_events8(word, T, S, kf=7)
    assert np.array_equal(ev["x"], x) and np.array_equal(ev["y"], y) and np.array_equal(ev["env"], env)
    assert np.array_equal(ev["substep"], sub) and np.array_equal(ev["p"], np.where(on == 1, 1, -1)) and np.all(ev["kf"] == 7)
    want_t = ((sub - 1) + (frac + 0.5) / 32768.0) * (T / S)
    assert np.abs(ev["t_off"].astype(np.float64) - want_t).max() < 1e-9
    assert np.all(ev["t_off"] > (sub - 1) * (T / S) - 1e-9) and np.all(ev["t_off"] < sub * (T / S) + 1e-9)


def test_bench_reads_the_committed_captures():
    """bench.py takes the step's instruction count and the chunk kernels' DRAM bytes from profiles/: the files must be
    there and parse (else the line silently loses `issue_roof` / `traffic`), and only for the workload they describe."""
    import bench
    cap = bench.range_capture(bench.RANGE_WORKLOAD)
    assert cap and 2.0e9 < cap["smsp__inst_executed.sum"] < 4.0e9          # warp-instructions per cfg 4 step
    assert cap["dram__bytes_read.sum"] > 1e9
    tr, rec = bench.step_traffic(bench.RANGE_WORKLOAD)
    assert tr and 5.0e9 < tr < 3.0e10                                       # one whole step: ~11 GB
    # the capture names the build it was taken on; `stale` compares that with the kernels in the tree
    assert rec["steps"] >= 2 and len(rec["csrc_sha"]) == 12 and rec["stale"] == (rec["csrc_sha"] != bench.csrc_sha())
    assert 2.0e9 < rec["warp_instructions_per_step"] < 4.0e9               # the same steps' instruction count (issue roof)
    for w in ("cfg2_16env_640x480_S16", "cfg3_64env_1280x720_S33_disk"):
        t2, r2 = bench.step_traffic(w)
        assert t2 > 1e9 and r2["events_per_step"] > 1e6
    assert bench.range_capture("cfg2_16env_640x480_S16") is None and bench.step_traffic("other") == (None, None)
    from paper_2607_08098_b200 import scenes
    assert {scenes.config(c).name for c in (2, 3, 4)} == set(bench.GRAPH_CAPTURES)
    peak, src = bench.hbm_peak()
    assert 3000.0 < peak < 9000.0 and src
