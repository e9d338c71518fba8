"""CPU oracle for the SOAP3-dp gapped-alignment stage (arXiv 1302.5507, Methods section 3).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package. It shares no
code with ``paper_1302_5507_b200`` and never imports it.
"""
from .oracle import (  # noqa: F401
    OracleScoring,
    OracleBatchResult,
    align_pair,
    align_batch,
    best_per_read,
    build,
    decode_cigar,
    mate_pairs,
    mate_windows,
    proper_pairs,
)
