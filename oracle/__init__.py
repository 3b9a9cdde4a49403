"""CPU oracle of the multispecies particle Landau scheme (arXiv:2212.00663).

TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  The product (paper_2212_00663_b200) never does.
"""
