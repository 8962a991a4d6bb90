"""CPU oracle (test infrastructure only; see oracle/gks_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2603_11102_b200.
"""
