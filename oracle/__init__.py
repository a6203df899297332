"""CPU oracle (test infrastructure only).  See oracle/coarse_oracle.c and oracle/oracle.py.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
"""
