"""B200-native synthetic Shack-Hartmann interaction-matrix engine (SynIM hot path).

``paper_2606_07759_b200.synim``      thin ctypes binding of the C-ABI library (CUDA, sm_100a)
``paper_2606_07759_b200.workloads``  seeded synthetic inputs (shared with the oracle; no method arithmetic)
"""
__all__ = ["workloads", "synim"]
