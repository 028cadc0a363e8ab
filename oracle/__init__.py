"""CPU oracle (test infrastructure).  See rms_oracle.c for the header and the list of pins.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
import this package.  It never imports paper_2012_06478_b200.
"""
from .rms_oracle import (  # noqa: F401
    build,
    philox4x32_10,
    direction,
    tables,
    step,
    init_walker,
    run,
    normalise,
    tensor_signal,
    volume_weighted_signal,
    OracleError,
)
