"""B200-native (sm_100a) MSD-AFQMC Wick's-theorem hot path (arXiv 2406.08314).

The product is the C-ABI library ``libmsd_b200.so`` (include/msd.h); this package is its thin Python
binding.  Import is lazy so that tools which only need the package path do not require the built
library; any call goes through the CUDA kernels and fails loudly if the library is missing.
"""
from .binding import (MSDError, MSDTrial, load_library, msd_force_bias, msd_force_bias_host, msd_greens,  # noqa: F401
                      msd_local_energy, msd_local_energy_host, msd_overlap, msd_overlap_host,
                      dist_allreduce, msd_setup, msd_setup_from_occ, setup_from_inputs)
from .binding import MSD_NOALLOC_SCRATCH_BYTES, MSD_OPT_3M_MAX_COND, MSD_OPT_COOP_MIN_ELEMS, MSD_OPT_NO_3M, MSD_OPT_NO_FUSED_S7, MSD_OPT_NO_SMEM_TILES  # noqa: F401

__all__ = ["MSDError", "MSDTrial", "load_library", "msd_setup", "msd_setup_from_occ", "msd_overlap",
           "msd_force_bias", "msd_local_energy", "msd_greens", "msd_overlap_host", "msd_force_bias_host",
           "msd_local_energy_host", "setup_from_inputs", "dist_allreduce", "MSD_OPT_NO_SMEM_TILES", "MSD_OPT_NO_FUSED_S7", "MSD_OPT_NO_3M",
           "MSD_OPT_COOP_MIN_ELEMS", "MSD_OPT_3M_MAX_COND", "MSD_NOALLOC_SCRATCH_BYTES"]
