"""fp64 CPU oracle for the bundle-adjustment LM/PCG hot path — TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this package.  It shares no code with `paper_2605_30583_b200` (the CUDA path)
and neither imports the other.
"""
from .binding import OracleBA, observation, rotation, spd_inverse, num_threads  # noqa: F401
