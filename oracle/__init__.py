"""CPU oracle for the SAGC rollout hot path.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
may import this package.  It shares no code with paper_2606_02218_b200 (the CUDA path)
and neither imports the other.
"""
