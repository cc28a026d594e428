"""B200-native Z4c RHS + Kreiss-Oliger + RK4 hot path of SACRA-K (arxiv/paper_2607_08743).

    from paper_2607_08743_b200 import sacra      # ctypes binding of libsacra (CUDA, sm_100a)
    from paper_2607_08743_b200 import workloads  # seeded synthetic inputs (numpy)

The binding fails loudly if the CUDA library is missing; there is no CPU fallback.
"""
__all__ = ["sacra", "workloads"]
