"""B200-native rand_cholQR with Count-Gauss multisketching (arxiv 2309.05868).

The product is the C-ABI library built from csrc/ (include/rqr.h); `binding` is the thin
Python marshalling layer over it.  Nothing here imports oracle/.
"""
__all__ = ["binding", "inputs", "flops"]
