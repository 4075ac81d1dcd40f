"""B200-native re-prefill hot path of SmoothAgent (arxiv/paper_2607_00151).

The product is ``libsmoothagent.so`` (C ABI in ``include/smoothagent.h``, CUDA kernels for sm_100a in
``csrc/``); ``binding`` exposes the same calls to Python, ``workloads`` generates the seeded synthetic
inputs, ``harness`` strings the calls together for tests and benchmarks.  No CPU fallback exists.
"""
from . import binding  # noqa: F401

__all__ = ["binding"]
