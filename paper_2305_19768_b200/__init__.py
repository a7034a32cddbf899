"""B200-native (sm_100a) hot path of pySecDec's numerical stage (arXiv:2305.19768):
randomly shifted rank-1 lattice evaluation of sector integrands, median lattice rule,
amplitude sum.  The compute lives in ``csrc/`` behind the C ABI of ``include/qmc.h``;
``binding`` is argument marshalling only.  Importing this package does not load the
CUDA library (``workloads`` must stay importable on a CPU-only box); the first call
into ``binding`` does, and fails loudly if it is missing.
"""
__all__ = ["workloads", "binding"]
