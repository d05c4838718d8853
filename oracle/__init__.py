"""CPU oracle for the DMRG hot path of arxiv 2503.20700 - TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.
It shares no code with paper_2503_20700_b200 (the CUDA path) and never imports it.
  fci.py   tier 1: brute-force full CI (plain definitions)
  dmrg.py  tier 2: plain block-sparse complementary-operator DMRG (H_eff x, renormalisation, sweep, RDMs)
"""
