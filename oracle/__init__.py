"""Float64 CPU oracle (TEST INFRASTRUCTURE -- see oracle/filark_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_2605_20132_b200.
"""
from .oracle import (BOX_DTYPE, EVENT_DTYPE, Oracle, OracleEma, OracleTrigger, build_oracle, oracle_associate, oracle_decimate,  # noqa: F401
                     oracle_zero_phase,
                     oracle_lib_path)
