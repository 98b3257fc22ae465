"""Oracle for the D3Q15 LBGK site update -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package. It shares no code with, and never
imports, ``paper_1906_11925_b200``. See ``hlb_oracle.cpp`` for what it computes.
"""
from .hlb_oracle import (  # noqa: F401
    Oracle,
    build,
    dense_run,
    velocity_set,
    run,
    VARIANT_SHIFTED,
    VARIANT_RAW,
    VARIANT_SHIFTED_LD,
    VARIANT_RAW_LD,
    LATTICE_Q,
    render,
    render_sample,
)
