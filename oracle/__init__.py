"""CPU oracle for the TDA Liouville operator of arXiv 2309.03513 (WEST-TDDFT).

TEST INFRASTRUCTURE ONLY.  This package is a plain, slow, FP64 numpy
restatement of what the hot path computes, written from the paper
(`PAPER.md` Eqs. 3, 4, 6, 8, 9 and 21, 23, 25) with the readings listed in
DESIGN.md.  It shares no code with the CUDA path and must never be imported
by the product (`paper_2309_03513_b200`); only `tests/`,
`__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference` legs of
`bench.py` may use it.

Parity status of each function is stated in its module header; the pins are
the `-m "not gpu"` tests under `tests/test_oracle_*.py`.  The paper prints no
worked numeric example of `AX`, so parity against paper-printed values is
unpinned; parity rests on closed forms, brute force and invariants.
"""
