"""Seeded synthetic inputs for the LST hot path (geometry tables and events).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2209_13711_b200/`).  It describes a detector and simulates
particles crossing it; it contains none of the method's arithmetic (no
mini-doublet / segment / triplet / quintuplet cuts, no module map, no fits).

Recipe: DESIGN.md "Synthetic inputs" (from BASELINE.json configs 1-5 and
SURVEY.md 8(d) / Appendix B).  Stands in for the CMS ttbar PU200 sample of
PAPER.md:103,139, which is not available.
"""
from .geometry import Geometry, build_geometry  # noqa: F401
from .events import Event, make_event, CONFIGS  # noqa: F401
