"""B200-native S2O4 gas-kinetic step with ALM + IBM forcing (arxiv/paper_2603_11102).

`gks` is the thin binding of the C-ABI library libgks_b200.so (hand-written sm_100a CUDA);
`workloads` holds the seeded synthetic inputs.  There is no CPU fallback.
"""
__all__ = ["gks", "workloads"]
