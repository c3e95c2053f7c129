"""B200-native CuBA hot path (arXiv:1208.0961): thin Python binding over the C-ABI library
`libcuba.so` (include/cuba.h).  Argument marshalling only -- every step of the path runs in
the hand-written sm_100a kernels under csrc/.  PyTorch supplies device memory and streams.

There is no CPU fallback: importing works anywhere (so the ABI can be inspected), but every
compute call needs the built library and a CUDA device and fails loudly otherwise.
"""
from .binding import (Cuba, CubaError, Counters, Trace, lib, lib_path, run_host,  # noqa: F401
                      workspace_bytes, launch_count, probe_fp64, strerror, EXPORTS,
                      observables_noalloc, NOALLOC_MAX_SLABS,
                      OPT_FUSE_HIST, OPT_GRAPH, OPT_SLOTS, OPT_SLOT_MARGIN)

from .slab import (SlabRank, LocalSlabGroup, slab_layers, layer_index, layer_weights, initial_selection, neighbours,  # noqa: F401,E402
                   exchange_halos, slab_step)

__all__ = ["SlabRank", "LocalSlabGroup", "slab_layers", "layer_index", "layer_weights", "initial_selection", "neighbours", "exchange_halos", "slab_step",
           "Cuba", "CubaError", "Counters", "Trace", "lib", "lib_path", "run_host",
           "workspace_bytes", "launch_count", "probe_fp64", "strerror", "EXPORTS", "observables_noalloc", "NOALLOC_MAX_SLABS",
           "OPT_FUSE_HIST", "OPT_GRAPH", "OPT_SLOTS", "OPT_SLOT_MARGIN"]
