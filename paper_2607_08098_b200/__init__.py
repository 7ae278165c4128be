"""EVIS per-pixel event-synthesis hot path for B200 (sm_100a); see DESIGN.md.

The CUDA library is loaded lazily by :mod:`paper_2607_08098_b200.binding`; importing the package
(e.g. for :mod:`scenes`, the seeded input generator) touches neither CUDA nor the oracle.
"""
__all__ = ["scenes", "binding", "build"]
