"""ORACLE — test infrastructure only: fp64 CPU implementation of the DLO-Lab rod step, written from the paper.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import this package.
"""
