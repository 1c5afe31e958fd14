"""CPU oracle of the ARGUS hot path — TEST INFRASTRUCTURE, NOT PRODUCT (see argus_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It shares no code with paper_2606_20374_b200 and imports nothing from it."""
from .oracle import (CELL_DTYPE, HEADER_DTYPE, SPAN_DTYPE, STAT_DTYPE, Oracle, build, bucket,
                     series)

from . import paper_literal  # noqa: F401  (the paper-literal float algorithms, NEXT-1..3)

__all__ = ["paper_literal", "CELL_DTYPE", "HEADER_DTYPE", "SPAN_DTYPE", "STAT_DTYPE", "Oracle", "build", "bucket",
           "series"]
