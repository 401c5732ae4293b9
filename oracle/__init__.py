"""ORACLE -- test infrastructure, NOT the product.

A plain, slow, CPU-only implementation of what the RT-TDA hot path computes, written from
PAPER.md (arXiv 2601.16949) and pinned by tests/ (`-m "not gpu"`) against closed forms, library
routines, invariants and the values the paper prints.  It shares no code with the CUDA path and
neither imports the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import it.

Parity status: every function is pinned; trajectories at configs 3-4
at the full step count are pinned only indirectly (prefix + operator parity), as DESIGN.md states.
"""
