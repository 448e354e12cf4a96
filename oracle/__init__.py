"""CPU oracle for the Concordia delta-checkpoint hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  The product (paper_2606_23521_b200) never does.
See oracle/concordia_oracle.c for what it follows in the paper and how it is pinned.
"""
from .oracle import (  # noqa: F401
    ORC_OK, ORC_ERR_INVALID, ORC_ERR_LOG_FULL, ORC_ERR_CORRUPT,
    Region, crc32c, crc32c_bitwise, scan, scan_mt, checkpoint, checkpoint_rle, checkpoint_marked, checkpoint_versions, apply_log, write_epoch, snapshot, compact_log, checkpoint_all, build,
)
