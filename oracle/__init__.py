"""fp64 CPU oracle for the MatrixFSDP owner-local optimizer step.

TEST INFRASTRUCTURE ONLY.  This package is the plain, slow, obviously-correct
restatement of what the hot path computes, written from /root/reference/PAPER.md
(arxiv/paper_2607_05895) and BASELINE.json's north_star.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs
may import it.  It shares no code with `paper_2607_05895_b200/` (the CUDA path)
and imports nothing from it.

Modules
  planner.py  Algorithm 1, roles, ROLE-/SCOPE-GREEDY, descriptor table.
  muon.py     momentum -> Frobenius normalisation -> K-step quintic Newton-Schulz -> update.
  adamw.py    decoupled-weight-decay Adam on packed tails.
  shampoo.py  owner-local Shampoo: L / R statistics, ridge, inverse fourth root by eigendecomposition,
              preconditioned update (readings S1-S5).

Pins (tests/test_oracle_*.py, `-m "not gpu"`): momentum closed form, SVD form of
the NS output, the quintic's band and printed scalar iterates, special matrices,
invariances, hand-computed update, AdamW two-step hand example, planner brute
force / Graham bound / hand traces; Shampoo: hand example, diagonal / orthogonal
closed forms, SVD form and polar-factor limit of the first step, P^4 S = I,
scipy's fractional_matrix_power, constant-gradient closed forms, invariances.  Unpinned: the planner against the *paper's
own* planner (the paper prints no assignment) -- "parity unpinned" for that one
comparison; see DESIGN.md section 4.
"""
