"""Seeded synthetic inputs shared by the tests, the benchmark and the oracle harness.

This package holds NONE of the imager's arithmetic (no indexing, no kernels, no gridding):
it only draws array layouts, uvw tracks, visibilities and weights with the shapes and value
distributions BASELINE.json's five configs state (recipe: DESIGN.md "Input recipe",
SURVEY.md section 8(d)).  Both `oracle/` and `paper_2206_15117_b200/` are fed from here;
neither is imported here.
"""
from .configs import CONFIGS, Workload, make_workload, uvw_tracks  # noqa: F401
