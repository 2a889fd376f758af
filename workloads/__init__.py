"""Seeded synthetic EPIC workloads (BASELINE.json configs C1..C5).

This module only *generates inputs*: antenna layouts, illumination-kernel tap
tables and channelised antenna voltages with the shapes and statistics of the
paper's LWA-SV data.  It holds none of the
method's arithmetic (no unpack, no gridding, no transform, no products) and is
imported by the tests, ``bench.py`` and ``__graft_entry__.smoke()`` to feed the
CPU oracle and the CUDA path the same bytes.  Neither ``oracle/`` nor the
``paper_1904_11422_b200`` package imports the other; both may import this.
"""
from .configs import (  # noqa: F401
    Workload,
    make_config,
    make_custom,
    make_lwa55,
    make_per_channel,
    pack_ci4,
    gaussian_taps,
    tophat_taps,
    CONFIG_NAMES,
)
