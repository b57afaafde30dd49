"""B200-native hot path of the hierarchical reduced-basis matched filter (arXiv:2110.13115).

`workloads` (seeded synthetic inputs) is importable without a GPU.  The CUDA path
lives behind the C-ABI library `librbmf.so` (csrc/, include/rbmf.h) and its thin
ctypes binding `paper_2110_13115_b200.rbmf`; importing the binding fails loudly when
the library has not been built (`python __graft_entry__.py` builds it).
There is no CPU fallback anywhere in this package.
"""

__all__ = ["workloads", "rbmf"]
