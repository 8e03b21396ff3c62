"""Seeded synthetic TPC time-frame generators.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
product (``paper_2009_07515_b200/``).  It holds none of the tracker's
arithmetic: it draws helix parameters from a counter-based RNG, intersects the
helices with the pad-row planes in double precision and emits fp32 SoA
clusters shaped like the workloads of BASELINE.json ``configs`` (PAPER.md:17,
29, 117-125: simulated Pb-Pb time frames at 50 kHz, pp at 0.2-1 MHz).
"""
from .generator import (  # noqa: F401
    Geometry,
    TimeFrame,
    CONFIGS,
    FOUR_REGION_PITCH,
    generate,
    generate_config,
    choose_cell,
    default_params,
    select_sectors,
    to_native_pad,
    to_native_time,
)
