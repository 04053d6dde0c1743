"""CPU oracle for the weighted-NMF hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  The product
(paper_2309_04623_b200) never does.
"""
