"""CPU oracle for the DNN-SP2-PT hot path (arXiv 2203.09621).  TEST INFRASTRUCTURE ONLY.

Plain, slow, fp64 numpy restatement of what the path computes, written from
/root/reference/PAPER.md (cited per function as PAPER.md:<line>).  It shares no
code with the CUDA path under `paper_2203_09621_b200/` and neither imports the
other; only `workloads/` (seeded inputs, no method arithmetic) serves both.

Only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference`
legs of `bench.py` may import this package.  The product never routes through it.

Parts:
  O1  closed_form.py   the DEFINITION: D0 = theta(mu I - H0), D1/D2 its directional
                       derivatives, by eigendecomposition.                 pinned
  O2  dnn_sp2_pt.py    the METHOD: Algorithms 1-3 step by step in fp64 (and, as
                       "O2-dh", with a numpy emulation of the dual-half product,
                       Eqs. 12-16 / 41-46).                                pinned
  O3  spectral.py      the same recursion on the eigenvalues only (control flow
                       cross-check, layer-count prediction at large N).    pinned

Pins live in tests/test_oracle_*.py (closed forms, finite differences, brute force,
invariants, special cases, block-matrix equivalence, the paper's printed 5e-5 / 1e-6
accuracy figures).  Parity unpinned: the layer counts and per-layer traces of the
paper's own runs (none are printed) and Table I (inputs unavailable).
"""
