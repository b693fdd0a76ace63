"""CPU oracle of the TemporalGS hot path -- TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs
may import this package.  The product path (`paper_2607_03390_b200`) never does.
"""
from .ora import Oracle, OraParams, OraStats, RECORD_DTYPE, build, lib  # noqa: F401
