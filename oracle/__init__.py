"""CPU oracle for the WPCD hot path -- TEST INFRASTRUCTURE ONLY (see wpcd_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.
"""
