"""pespace-b200: B200-native batched detector response + Whittle likelihood (arxiv 2602.12011).

Public API (thin ctypes binding over the C ABI of include/pespace.h):
    response, loglike, fisher        -- device tensors in, device tensors out
    loglike_host                     -- host numpy buffers, copies inside the call
The CUDA library is mandatory: importing `paper_2602_12011_b200.binding` fails loudly when
libpespace.so has not been built (python -m paper_2602_12011_b200.build).  There is no
CPU fallback.
"""
__all__ = ["workloads"]
