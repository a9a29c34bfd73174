"""CPU oracle of the Hough track-finding path -- TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py` (cpu_baseline / --impl reference) may import
this package.  `paper_1311_2769_b200` never does; the two share no code.
"""
from .binding import (Oracle, OracleCandidates, CAND_DTYPE)  # noqa: F401
