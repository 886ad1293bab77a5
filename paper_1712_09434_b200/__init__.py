"""B200-native TPC sector tracker (arXiv:1712.09434 section 3): thin Python binding of
``include/tpc_tracker.h``.  Every step of the path runs in the CUDA kernels of
``csrc/``; this package only marshals arguments.  There is no CPU fallback: importing
works without a GPU (so that the exported symbols can be checked), any compute call
without the extension or without a device raises.
"""
from .binding import (  # noqa: F401
    Tracker, TrackerParams, TrackResult, MergedResult, ClusterTransform, ItsTracker, slice_frames, slice_frames_static, slice_static_setup, SLICE_STATIC_MAX_ENTRIES, TpcError, load_library, library_path, exported_symbols,
    STATUS_TRACKLET_OVERFLOW, STATUS_TRACK_OVERFLOW, STATUS_HIT_OVERFLOW, COUNTER_NAMES,
)
from .sharding import shard_events  # noqa: F401
