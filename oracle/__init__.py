"""CPU oracle for the channel-flow DNS substep of arxiv 1808.06461 (section 2.1, 3.2).

TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 numpy restatement of what the hot path computes,
written from PAPER.md and the readings listed in DESIGN.md ("Readings of the paper").  It shares
no code, tables or helpers with the CUDA path under ``paper_1808_06461_b200/`` and must never be
imported by it: only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.

Parity status: every function is pinned by ``tests/test_oracle_*.py`` (``-m "not gpu"``) against
closed forms, brute force or analytic solutions, EXCEPT the paper's own optimised "spectral-like"
compact coefficients and its optimised wall mesh, which the paper does not
print: **parity unpinned** against the paper's production code for those two items; the oracle uses
the maximal-order rows of DESIGN.md reading R4 instead.
"""
