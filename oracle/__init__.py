"""CPU oracle of the TPC sector tracker — test infrastructure only (see tpc_oracle.cpp header)."""
from .oracle import (COUNTER_NAMES, DEFAULT_CUTS, MODE_GRID, MODE_ROWSCAN, MODE_TRIPLET, TRACK_DTYPE, Oracle,
                     OracleResult, build)

__all__ = ["COUNTER_NAMES", "DEFAULT_CUTS", "MODE_GRID", "MODE_ROWSCAN", "MODE_TRIPLET", "TRACK_DTYPE", "Oracle",
           "OracleResult", "build"]
