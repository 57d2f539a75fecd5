"""CPU oracle of the SPH pipeline of arXiv 2110.02621 — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  The product (paper_2110_02621_b200) never does.
"""
