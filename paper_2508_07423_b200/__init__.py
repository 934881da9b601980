"""B200-native hits -> edge-scores path of the ETX4VELO GNN tracking pipeline (arXiv 2508.07423).

Sub-modules
-----------
synth    seeded synthetic inputs (events, weights, configs); holds none of the method's arithmetic
binding  ctypes binding of the C-ABI library ``libetx.so`` (include/etx.h); argument marshalling only
build    nvcc build of ``csrc/`` into ``libetx.so`` (sm_100a)

Nothing is imported eagerly: ``synth`` must stay importable without the CUDA library, and
``binding`` must fail loudly (never fall back) when the library is missing.
"""

__all__ = ["synth", "binding", "build"]
