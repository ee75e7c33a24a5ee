"""Seeded synthetic inputs for the UT decode + Compass path.

This package is the ONLY code shared by the CPU oracle (``oracle/``) and the
CUDA product (``paper_2002_11529_b200/``).  It holds input generation and the
truth bookkeeping used to score results -- none of the method's arithmetic:
no raw-bank decoding, no window search, no fit.  It stands in for the LHCb
Monte-Carlo samples (minbias, Bs->phiphi), the UT geometry
tables and the raw-bank format, which are not available.
The recipe is SURVEY.md section 8(d) / BASELINE.json ``configs``; DESIGN.md
section 4 restates it.
"""
from .geometry import UTGeometry, make_geometry
from .events import EventModel, Batch, generate_batch, generate_event, encode_event
from .configs import CONFIGS, WorkloadConfig, CompassParams, make_compass_params, make_workload
from .truth import physics_metrics
from .field import KickLUT, make_kick_lut

__all__ = [
    "UTGeometry", "make_geometry", "EventModel", "Batch", "generate_batch",
    "generate_event", "encode_event", "CONFIGS", "WorkloadConfig", "CompassParams",
    "make_compass_params", "make_workload", "physics_metrics", "KickLUT", "make_kick_lut",
]
