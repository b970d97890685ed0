"""B200-native near-field direct gravity sum (the Abacus near field of arXiv:2110.11398).

The product is ``libnf_b200.so`` -- hand-written CUDA for sm_100a behind the C-ABI declared in
``include/nf.h``.  This package is its thin Python binding.  Importing it loads (and, if stale and
nvcc is present, rebuilds) the library; without it the import fails: there is no CPU path.
"""
from .binding import (  # noqa: F401
    Plan, NFError, LIB_PATH, EXPORTS,
    nf_plan_create, nf_bin, nf_rebin, nf_accel, nf_accel_density, nf_accel_kick, nf_set_masses, nf_set_sink_slabs, nf_destroy, nf_bin_host, nf_accel_host, nf_last_error,
    nf_set_stream, nf_workspace_bytes, nf_set_workspace, nf_get_binning, nf_get_layout, nf_get_stats,
    nf_set_option, nf_slab_histogram, nf_slab_histogram_static, nf_slab_select, nf_get_slab_cost, nf_slab_partition,
)
