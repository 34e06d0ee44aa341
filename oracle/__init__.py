"""ORACLE — test infrastructure, not the product (see adept_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2302_08252_b200``.
"""
from .binding import Oracle, build, lib, math_fns, TRACE_DTYPE  # noqa: F401
