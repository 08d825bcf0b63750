"""B200-native arrested-Newton-flow hot path of arxiv/paper_2603_24370 (soliton_solver).

`paper_2603_24370_b200.ss`        thin ctypes binding of the C-ABI library libss.so (CUDA, sm_100a)
`paper_2603_24370_b200.workloads` seeded synthetic inputs (numpy only; shared with the oracle tests)

Nothing here falls back to the CPU: importing `ss` without the built library raises.
"""
__all__ = ["workloads"]
