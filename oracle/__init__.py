"""oracle/ -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain CPU statement of what the hot path of arXiv 1603.08357 computes (see ccl_oracle.c and
komura_steps.py).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package; paper_1603_08357_b200/ never does.
"""
