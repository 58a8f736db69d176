"""Seeded synthetic input generator (no method arithmetic; see synth.py)."""
from .synth import (DEFAULT_SEED, Workload, make_workload, eval_points, floating_start,  # noqa: F401
                    amplitudes, angular, cnormal, uniform, build)
