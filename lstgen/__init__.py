"""Seeded synthetic-input generators for the LST hot path (geometry, events, DNN weights).

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA path
(`paper_2403_13166_b200/`).  It contains none of the method's arithmetic: no
mini-doublet / segment / triplet / quintuplet cut, no DNN evaluation, no pLS matching.
It only fabricates inputs with the shapes and distributions of BASELINE.json `configs`
(recipe: DESIGN.md "Input recipe", SPEC.md section 2).
"""
from .geometry import Geometry, build_geometry
from .events import Event, make_event, config_event, CONFIG_SEEDS
from .weights import xavier_weights, N_WEIGHTS, N_FEAT, N_HID

__all__ = [
    "Geometry", "build_geometry", "Event", "make_event", "config_event", "CONFIG_SEEDS",
    "xavier_weights", "N_WEIGHTS", "N_FEAT", "N_HID",
]
