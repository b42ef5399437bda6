"""Seeded synthetic input generators shared by the oracle, the CUDA path's tests and bench.py.

This package builds INPUTS only: chirp templates, the time-slice layout, the per-slice SVD bank
(the offline step of PAPER.md:112-119 that the hot path takes as its argument) and white-noise
strain with injections.  It holds none of the hot path's arithmetic (no resampling, no filtering,
no reconstruction, no peak search) and imports neither ``oracle`` nor ``paper_2511_04730_b200``.
"""
from .lloid_inputs import (  # noqa: F401
    Bank,
    Slice,
    Injection,
    chirp_templates,
    chirp_time_to_merger,
    chirp_frequency,
    slice_layout,
    build_bank,
    bank_from_layout,
    slice_template_matrices,
    decompose_slice,
    injection_waveform,
    random_bank,
    random_triggers,
    template_autocorrelations,
    make_strain,
    inject,
    make_config,
    CONFIGS,
)
