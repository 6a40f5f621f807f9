"""pct-b200: single-B200 proton-CT hot path (MLP -> rows of A -> block-iterative DROP).

Sub-modules
  binding  thin ctypes binding of the C-ABI in include/pct.h (libpct.so; fails loudly if missing)
  build    in-tree nvcc build of csrc/ for sm_100a
  regions  Algorithm 1 of the paper across processes (one z-region per GPU; torch.distributed plumbing only)
"""
__all__ = ["binding", "build", "regions"]
