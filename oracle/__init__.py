"""ORACLE — test infrastructure, NOT product code.

A plain, slow, obviously-correct CPU implementation (Python + numpy, fp64) of what the prefix-cached
prefill path computes, written from PAPER.md (arxiv/paper_2606_19667, CacheWeaver) and the readings listed in
DESIGN.md.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
import it.  It shares no code with paper_2606_19667_b200/ and never imports it; the product never imports
this package.  Pinned by `pytest -m "not gpu"` (tests/test_oracle_*.py); timing claims: "parity unpinned"
(the paper prints no kernel time).
"""
