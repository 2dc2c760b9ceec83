"""fp64 CPU oracle for the bundle-adjustment LM/PCG hot path — TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this package.  It shares no code with `paper_2605_30583_b200` (the CUDA path)
and neither imports the other.
"""
from .binding import (OracleBA, num_threads, observation, observation_model, retract_camera, rotation,  # noqa: F401
                      spd_inverse)
