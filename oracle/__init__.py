"""fp64 CPU oracle for the TDGL hot path of arXiv:1409.8340.

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (`paper_1409_8340_b200/`,
`include/`) may import, call, link or execute anything in this package; only
`tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs do.  It shares no code with the CUDA path.
"""
