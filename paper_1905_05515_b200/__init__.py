"""paper_1905_05515_b200 -- B200-native TPC sector track finding (CA seeding + Kalman tracklets + selector).

Thin Python binding over the C ABI of include/tpc.h (libtpc_b200.so, hand-written CUDA for sm_100a).  Argument marshalling
only: every step of the path runs in the library's kernels.  There is no CPU fallback; without the built library or
without a CUDA device the calls raise.
"""
from .binding import (TpcError, Tracker, Tracks, abi_symbols, lib_path, load_library,  # noqa: F401
                      tpc_create, tpc_load_clusters, tpc_load_clusters_batch, tpc_find_tracks, tpc_find_tracks_device,
                      tpc_refit_tracks, tpc_mark_clusters, tpc_merge_tracks, tpc_find_loopers, tpc_find_loopers_noalloc, tpc_clear, tpc_destroy, tpc_set_param, tpc_set_stream, tpc_get_timings)
from .sharding import shard_units  # noqa: F401
