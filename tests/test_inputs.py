"""Seeded input generators (no GPU): the threshold maps handed to evis_set_thresholds (Eq. 8)."""
import numpy as np

from paper_2607_08098_b200 import scenes


def test_threshold_maps_follow_the_stated_draw():
    """theta ~ max(N(C, sigma^2), theta_min) once per pixel: right mean and spread, the
    floor is respected, ON and OFF maps are different draws, and the maps are reproducible."""
    spec = scenes.small(scenes.config(3), num_envs=2, height=120, width=160)         # C+ = 0.2, C- = 0.3
    on, off = scenes.threshold_maps(spec, sigma=0.03, theta_min=0.01)
    on2, off2 = scenes.threshold_maps(spec, sigma=0.03, theta_min=0.01)
    assert on.shape == off.shape == (2, 120, 160) and on.dtype.is_floating_point
    assert np.array_equal(on.numpy(), on2.numpy()) and np.array_equal(off.numpy(), off2.numpy())
    assert abs(float(on.mean()) - spec.c_pos) < 2e-3 and abs(float(off.mean()) - spec.c_neg) < 2e-3
    assert abs(float(on.std()) - 0.03) < 3e-3 and abs(float(off.std()) - 0.03) < 3e-3
    assert abs(float(np.corrcoef(on.numpy().ravel(), off.numpy().ravel())[0, 1])) < 0.05
    lo, _ = scenes.threshold_maps(spec, sigma=0.5, theta_min=0.05)
    assert float(lo.min()) == np.float32(0.05) and float((lo == np.float32(0.05)).float().mean()) > 0.2
