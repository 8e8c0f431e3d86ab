"""CPU oracle for the WP-CCC hot path (arXiv 2403.04252).

TEST INFRASTRUCTURE ONLY.  A plain, slow, fp64 numpy restatement of what the hot path
computes, written from the paper in the paper's order and notation, with the
readings of SURVEY.md §8(c) / DESIGN.md.  It shares no code with the CUDA library in
``paper_2403_04252_b200/`` and neither imports the other.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import it.

Pins (tests/test_oracle_*.py, -m "not gpu"): every function below is pinned to closed
forms, library routines (sympy / scipy), brute force or invariants; see DESIGN.md §Oracle.
Numeric parity *with the paper* is unpinned: the paper prints no worked example
(PAPER.md contains ratios only).
"""
