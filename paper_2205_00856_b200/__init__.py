"""B200-native N-shaped partition Crank-Nicolson stepper (arxiv 2205.00856): C-ABI library + thin binding.

`from paper_2205_00856_b200 import binding` loads libcn_nshape.so on first use and fails loudly if it is
missing; `workloads` holds the seeded synthetic inputs and none of the method's arithmetic.
"""
__all__ = ["binding", "workloads", "build"]
