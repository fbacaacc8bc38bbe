"""CPU oracle for the TPC CA track finder (TEST INFRASTRUCTURE -- see tpcca_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from the CUDA path.
"""
from .oracle import DEFAULT_MERGE_PARAMS, DEFAULT_PARAMS, DEFAULT_TIME_PARAMS, OracleResult, build, kf_transport, kf_update, refit_hits, rotate_frame, time_estimate_state, track  # noqa: F401
