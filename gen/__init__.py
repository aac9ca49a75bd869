"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds NO arithmetic of the TRED method (no drift, no charge
density, no quadrature, no convolution): it only draws random track
geometry, charges and a synthetic field response, and carries the plain-data
configuration record.  See DESIGN.md "Input recipe".
"""
from .workloads import (Config, make_config, make_segments, make_response,
                        make_random_response, SEG_FIELDS, make_steps, STEP_FIELDS, STEP_PARAMS)

__all__ = ["Config", "make_config", "make_segments", "make_response",
           "make_random_response", "SEG_FIELDS", "make_steps", "STEP_FIELDS", "STEP_PARAMS"]
