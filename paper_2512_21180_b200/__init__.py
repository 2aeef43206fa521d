"""B200-native cone-beam CT projector / backprojector (LIRE++ hot path).

`paper_2512_21180_b200.cbct` is the thin ctypes binding over the C ABI in
`include/cbct.h` (libcbct.so, hand-written CUDA for sm_100a);
`paper_2512_21180_b200.synth` holds seeded synthetic workloads;
`lire_ops` walks the operator calls of Algorithm 1 over the three scales and
`autograd` wraps the projector pair for `torch.autograd` (both import torch).
"""
__all__ = ["cbct", "synth"]
