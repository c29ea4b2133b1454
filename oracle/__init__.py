"""CPU oracle for the FlashCP hot path (arxiv/paper_2606_08476).

TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct numpy code (integers for the
planner and index sets, fp64 for attention) written from PAPER.md.  It shares no code with
the CUDA path in ``paper_2606_08476_b200/`` and neither imports the other.  Only ``tests/``,
``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs of
``bench.py`` may import it.

Modules
-------
planner    Algorithm 1 in the deterministic reading of DESIGN.md section 3.
kvselect   sharding-aware KV selection, Eq. 4 / Eq. 5.
attention  document-masked causal attention forward/backward and the
           partial-result (LSE) merge.

Pin status (see tests/test_oracle_*.py; every function below has a pin that is not itself):
  planner.W .................. brute-force pair count
  planner.plan ............... hand-worked examples under tests/golden/, Eq.1/Eq.2 invariants,
                               Per-Doc pair identity, brute-force optimum lower bound.
                               PARITY UNPINNED against the *authors'* implementation: the paper's
                               Table 2 (28 % / 1.04) needs Pile and their code.
  kvselect.* ................. pair-by-pair brute force of the needed-key set, Eq.5 <= Eq.4
  attention.* ................ triple-loop brute force, torch SDPA special case, closed forms
                               (K=0 -> lse = ln(#visible keys)), plan invariance, merge identity,
                               central finite differences.
"""
