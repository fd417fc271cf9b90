"""Oracle package: TEST INFRASTRUCTURE ONLY (see gbees_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this. The product package never does.
"""
