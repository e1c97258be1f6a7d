"""B200-native batched quadrotor simulation step (Crazyflow hot path, arxiv/paper_2606_01478).

`paper_2606_01478_b200.cf` is the thin Python binding over the C-ABI library `libcf.so`
(include/cf.h); `paper_2606_01478_b200.workloads` holds the seeded synthetic input recipes.
Nothing here falls back to a CPU path: importing `cf` without the built CUDA library raises.
"""
__all__ = ["workloads"]
