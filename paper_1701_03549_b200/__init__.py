"""libfire for NVIDIA B200: batched stochastic cellular-automata fire propagation + fitness reduction,
the hot path of arXiv 1701.03549 (Denham & Laneri).  See DESIGN.md and include/fire.h.

    from paper_1701_03549_b200 import libfire     # C-ABI binding (CUDA only, no CPU fallback)
    from paper_1701_03549_b200 import workloads   # seeded synthetic inputs (no method arithmetic)
"""
__all__ = ["libfire", "workloads", "build"]
