"""CPU oracle for the TPC CA track finder (TEST INFRASTRUCTURE -- see tpcca_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from the CUDA path.
"""
from .oracle import (DEFAULT_LEG_FIT_PARAMS, DEFAULT_LEG_PARAMS, DEFAULT_MERGE_PARAMS, DEFAULT_PARAMS, DEFAULT_TIME_PARAMS, TAG_EXTRA_LEG,  # noqa: F401
                     TAG_HIGH_INCLINATION, TAG_LOW_PT, OracleResult, angle_upper, build, kf_transport, kf_update, leg_end,
                     leg_pair, refit_hits, rotate_frame, time_estimate_state, track)
