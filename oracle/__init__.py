"""CPU oracle for the OPTCC hot path (arxiv/paper_2606_01680) -- TEST INFRASTRUCTURE ONLY.

Plain, slow, obviously-correct Python/numpy written from /root/reference/PAPER.md and
docs/PLAN_SPEC.md.  It shares no code with the CUDA/C++ library under
paper_2606_01680_b200/ and never imports it.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import it; the product path never does.

Modules
  closed_forms  T0, Theorems 1/2/3/6/13, Eq.(1)/(2), App. C/D.3/E.4 forms      (pinned)
  planner       canonical plan tables of docs/PLAN_SPEC.md                       (pinned)
  interpreter   walks a plan: contributor sets, hazards, fp32/bf16 plan-order emulation (pinned)
  cost_sim      port-model event simulation in exact rationals                   (pinned)
  reference     fp64 per-element reference sum and the tolerance predicates      (pinned)
  brute_force   exhaustive search over chunk splits for p <= 5                   (pinned)
  cwalk/walk.c  interpreter.run_f32 restated in plain C (OpenMP over the independent flows of a
                step): the compiled CPU baseline bench.py times; pinned against run_f32 bit for bit

Parity unpinned: the slot-exact pattern layouts of Figs 5-7, 11-19 (figures absent from
PAPER.md); they are replaced by the canonical constructions of docs/PLAN_SPEC.md, which are
pinned through the paper's closed-form times, flow counts and invariants instead.
"""
