"""B200-native Trotter-Suzuki spin-1/2 time step (arXiv:1305.0036).

`workloads` (seeded inputs) has no dependency on the CUDA library; `binding` loads
`libts_b200.so` lazily on first use and fails loudly if it is missing.
"""
__all__ = ["binding", "workloads"]
