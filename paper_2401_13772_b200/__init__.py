"""B200-native SP2 density-matrix purification (arxiv 2401.13772 hot path).

The compute path is the C-ABI library ``libbmlsp2.so`` (hand-written sm_100a CUDA, ``csrc/``); ``api`` is the thin
ctypes binding with the same entry-point names.  Nothing here falls back to the CPU: importing ``api`` without the
built library raises.
"""
__all__ = ["api", "hamiltonians"]
