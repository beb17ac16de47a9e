"""fp64 CPU oracle (TEST INFRASTRUCTURE). See oracle/nasg_ref.c, oracle/sh_ref.c, oracle/ref.py.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package. The product package never does.
"""
