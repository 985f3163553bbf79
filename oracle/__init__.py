"""fp64 single-threaded CPU oracle of the PIC particle step — TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with, and never
imports, ``paper_2110_08650_b200``; the product never imports it.
Definitions: SURVEY.md §8(c) steps 1-7 (the paper, names none of them).
"""
from .pic_oracle import (  # noqa: F401
    OracleParams,
    build,
    boris,
    deposit,
    gather,
    lib,
    move,
    rho,
    shape,
    step,
    wrap_and_bucket,
    Oracle,
)
from . import yee_oracle  # noqa: F401,E402  (field update)
