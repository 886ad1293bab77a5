"""Seeded synthetic TPC events (inputs only).

This package is the ONE thing the CPU oracle (``oracle/``) and the CUDA path
(``paper_1712_09434_b200/``) have in common: it draws the input clusters.  It
contains none of the tracker's arithmetic (no grid, no chi2, no Kalman
filter) - only the detector geometry of BASELINE.json's configs and an exact
fp64 helix that is sampled, smeared and cast to fp32.
"""
from .events import (  # noqa: F401
    Geometry,
    EventSpec,
    ClusterBatch,
    CONFIGS,
    default_geometry,
    generate_event,
    generate_config,
    generate_tracks_event,
    concat_batches,
    take_tasks,
)
from .calibration import RawCalibration, default_calibration, raw_from_yz  # noqa: F401
from .frames import make_frame  # noqa: F401
from .its import ItsGeometry, ItsBatch, default_its_geometry, generate_its_events  # noqa: F401
