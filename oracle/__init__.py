"""fp64 CPU oracle of the DAO hot path -- TEST INFRASTRUCTURE (see dao_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package; the product path never does.
"""
