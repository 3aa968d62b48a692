"""Harness code shared by tests/, bench.py and __graft_entry__.smoke(): the seeded synthetic input generator
(:mod:`harness.synth`, ground-truth motion model only: none of the method's arithmetic), the algorithmic
flop/byte model behind the roofline numbers (:mod:`harness.workmodel`) and the replicas-only multi-GPU helpers
(:mod:`harness.replicas`).  Not part of the product library (paper_2603_25834_b200/)."""
