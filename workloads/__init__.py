"""Seeded synthetic inputs for the cuHARM hot path ("Input recipe").

This package serves BOTH the CPU oracle's tests and the CUDA path's tests / bench.  It holds
parameter dictionaries and initial-data generators only; it imports neither `oracle` nor
`paper_2205_02484_b200`, and neither of them imports it for anything but inputs.
"""
from .params import default_params, config, r_horizon, SEED  # noqa: F401
