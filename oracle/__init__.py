"""CPU oracle of the checkerboard Metropolis sweep (arXiv 1411.0127).  TEST INFRASTRUCTURE ONLY.

May be imported only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  Shares no code with paper_1411_0127_b200/ (the CUDA path).
"""
