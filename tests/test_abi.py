"""CPU-only checks of the boundary: libevis.so builds for sm_100a, loads, exports every symbol that
include/evis.h declares, and rejects bad arguments without touching a GPU."""
import ctypes as C
import os
import re

import pytest

from paper_2607_08098_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def _declared():
    src = open(os.path.join(ROOT, "include", "evis.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(evis_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert {"evis_create", "evis_step", "evis_read_events", "evis_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"libevis.so lacks {n}"
    assert sorted(binding.SYMBOLS) == names


def test_struct_layouts_match_the_header():
    assert C.sizeof(binding.evis_config) == 64
    assert binding.EVENT_DTYPE.itemsize == 16
    assert C.sizeof(binding.evis_info) == 80


def test_argument_validation_needs_no_gpu(lib):
    ctx = C.c_void_p()
    assert lib.evis_create(None, C.byref(ctx)) == binding.EVIS_ERR_INVALID_ARG
    good = dict(num_envs=1, height=8, width=8, substeps=4, c_pos=0.2, c_neg=0.2, log_eps=1e-3,
                keyframe_dt=1 / 60, max_motion_px=0.0, composite_mode=0, path=0, device=0,
                event_capacity=1024, debug_capture=0, reserved=0)
    for bad in (dict(num_envs=0), dict(height=-1), dict(width=40000), dict(substeps=0), dict(substeps=256),
                dict(c_pos=0.0), dict(c_neg=-1.0), dict(log_eps=0.0), dict(keyframe_dt=0.0),
                dict(composite_mode=7), dict(path=9), dict(event_capacity=0), dict(max_motion_px=-1.0),
                dict(c_pos=float("nan"))):
        cfg = binding.evis_config(**{**good, **bad})
        assert lib.evis_create(C.byref(cfg), C.byref(ctx)) == binding.EVIS_ERR_INVALID_ARG, bad
        assert not ctx.value
    assert lib.evis_step(None, None, None, None, None, None, None) == binding.EVIS_ERR_INVALID_ARG
    assert lib.evis_read_events(None, None, 0, 0, None) == binding.EVIS_ERR_INVALID_ARG
    assert lib.evis_get_info(None, None) == binding.EVIS_ERR_INVALID_ARG
    assert lib.evis_set_env_offset(None, 0) == binding.EVIS_ERR_INVALID_ARG
    assert lib.evis_destroy(None) == binding.EVIS_OK
    assert lib.evis_strerror(binding.EVIS_ERR_OVERFLOW) == b"event capacity exceeded"
    assert b"sm_100a" in lib.evis_version()


def test_product_path_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import or reference it."""
    pkg = os.path.join(ROOT, "paper_2607_08098_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "evis_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f
