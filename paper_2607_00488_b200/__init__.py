"""B200-native spectrum-reweighting likelihood hot path (arxiv/paper_2607_00488).

The compute path lives in csrc/ (hand-written sm_100a CUDA behind the C ABI of
include/rw.h); `binding` is argument marshalling only.  Importing the package does not
load the CUDA library; the first call does, and fails loudly if it is missing.
"""
__all__ = ["binding", "workloads"]
