"""Seeded synthetic inputs for the EMC hot path (shared by tests, bench.py and the oracle leg).

This package holds NO arithmetic of the method itself: everything is numpy's seeded random number
generator plus library routines (numpy.fft, scipy.spatial.transform.Rotation,
scipy.ndimage.map_coordinates).  Neither `oracle/` nor `paper_1409_4256_b200/` is imported here.
The recipe is stated in DESIGN.md ("Input recipe").
"""
from .synth import (  # noqa: F401
    CONFIGS,
    EmcConfig,
    EmcInputs,
    blob_object,
    detector_geometry,
    detector_mask,
    intensity_model,
    ladder_rotations,
    make_inputs,
    random_rotations,
    rotation_ladder,
    simulate_patterns,
)
