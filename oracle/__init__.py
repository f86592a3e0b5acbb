"""CPU oracle of the STREAmS-2 hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares nothing with paper_2304_05494_b200.
"""
