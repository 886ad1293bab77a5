"""CPU oracle of the TPC sector tracker - TEST INFRASTRUCTURE ONLY.

Importable from ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
cpu_baseline / ``--impl reference`` legs; never from ``paper_1712_09434_b200``.
"""
from .oracle import (  # noqa: F401
    OracleParams, OracleResult, track, transport, update, COUNTER_NAMES, canonical_tracks,
    MergeResult, merge_refit, rotate, refit_hits,
)
