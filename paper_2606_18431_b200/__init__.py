"""UniBoost scheduling-step simulator for B200 (sm_100a): Python binding of libuniboost.so.

The library is loaded lazily on first use and fails loudly if it is missing;
there is no CPU fallback.  `workloads` (seeded input generators) imports numpy only.
"""
__all__ = ["workloads"]
