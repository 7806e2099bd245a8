"""CPU oracle for the BTA / INLA value-and-gradient hot path.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this package.  It shares no code with `paper_2605_06392_b200/` (the CUDA
path) and never imports it; both consume the arrays made by `workloads/`.
"""
