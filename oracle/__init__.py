"""CPU ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, obviously-correct CPU implementation of what the hot path of
AnchorTP's state-preserving recovery computes (§III-B/C, Alg. 1,
Eq. 1, Fig. 3), written from the paper.  It shares no code with the CUDA
library under ``paper_2511_11617_b200/`` and neither imports the other; only
``workloads/`` (input shapes + seeded byte generators, no method arithmetic)
serves both.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import, call, link or execute anything here.

Modules (each function cites the passage it follows):
  planning.py    S1 partition (Alg.1 l.2-5), S2 CMM (Alg.1), Eq.1 bound,
                 Greedy / Full-Reload comparison planners
  bruteforce.py  exhaustive minimum over all per-unit source assignments (tiny instances)
  state.py       slot addressing, plan application to parameter slabs and paged KV
                 (element by element, via etp_apply.c), page-table rule, plain definitions
  etp_apply.c    the element-by-element loops (plain C, -O2, no intrinsics)
  linear.py      unsharded Y = X W^T reference (fp64)

Pin status (tests/test_oracle_*.py, all ``-m "not gpu"``):
  partition      pinned: Fig. 3 bounds 0/341/682/1024; widths in {floor, ceil}, sum = S (:94)
  cmm_plan       pinned: Fig. 3 task list; Eq. 1 closed form (:156); brute force on tiny
                 instances; invariants I1-I5; Table II ordering in units (:204)
  apply_params   pinned: plain definition (new shard == slice of the unsharded tensor), untouched bytes,
                 hand-written golden slab image (tests/golden/slab_tiny.txt)
  apply_kv       pinned: plain definition KV_ref[s][t][l][c][h] readable at its new place (numpy N-d views, not the
                 oracle's offset arithmetic); hand-written golden tests/golden/kv_tiny.txt (relocated block, TRANSFER
                 head, RELOAD head into a wrapped slot, both layouts; tests/test_oracle_state.py::test_golden_kv_image)
  page_table     pinned: hand-worked example (tests/golden/page_table.txt), injectivity / budget properties.
                 The eviction + relocation RULE itself is a DESIGN.md reading (K5) of PAPER.md:86 — the
                 paper fixes only "LRU"; no value in the paper pins the relocation order.
  linear_ref     pinned: textbook definition checked against an explicit triple loop
"""
