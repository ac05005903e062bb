"""B200-native SOP overdamped-Langevin hot path (arxiv 1003.1148): thin Python binding over the C ABI in
include/sop.h.  All computation runs in the CUDA kernels of csrc/; PyTorch only provides device memory and the
stream.  There is no CPU fallback: importing `sop` without a loadable libsop.so raises."""
from .sop import (Sop, SopError, sop_create, sop_run, sop_sync, sop_get_coords, sop_set_coords, sop_get_energies,
                  sop_get_forces, sop_get_lists, sop_get_step, sop_set_step, sop_destroy, from_workload,
                  library_path, exported_symbols)
from .sharding import shard_trajectories

__all__ = ["Sop", "SopError", "sop_create", "sop_run", "sop_sync", "sop_get_coords", "sop_set_coords",
           "sop_get_energies", "sop_get_forces", "sop_get_lists", "sop_get_step", "sop_set_step", "sop_destroy",
           "from_workload", "shard_trajectories", "library_path", "exported_symbols"]
