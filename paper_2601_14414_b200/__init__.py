"""pimpc-b200: sm_100a CUDA implementation of the piMPC accelerated/restarted ADMM iteration
(arxiv 2601.14414, Algorithm 1) behind the C ABI declared in include/pimpc.h.

`workloads` (seeded input generators) imports without the CUDA library; `pimpc` (the binding)
fails loudly if libpimpc.so is missing -- there is no CPU fallback.
"""
__all__ = ["workloads"]
