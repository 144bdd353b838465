"""B200-native (sm_100a, FP64) GP prediction pipeline of arxiv/paper_2602_19683.

The product is the C-ABI library declared in include/gp_b200.h (built from csrc/ into
libgp_b200.so); `binding` is the thin argument-marshalling layer over it and `nfir` the
seeded synthetic input generator.  Nothing is imported eagerly so that `nfir` can be used
without the CUDA library (it holds none of the method's arithmetic).
"""
__all__ = ["binding", "nfir", "build"]
