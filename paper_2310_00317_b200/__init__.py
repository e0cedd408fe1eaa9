"""B200-native multi-turn single-particle tracking (the hot path of arxiv 2310.00317).

The product is the C-ABI library ``libxt_b200.so`` (``include/xt.h``); this package holds
its CUDA sources (``csrc/``), the in-tree nvcc build (``_build``) and a thin ctypes binding
(``binding``) whose functions carry the names of the C entry points.  It never imports
``oracle`` (test infrastructure) and has no CPU fallback.
"""
from .binding import (  # noqa: F401
    XtError, Lattice, load_library, new_particles, particles_to_device, particles_to_host,
    xt_lattice_create, xt_lattice_create_ex, xt_lattice_destroy, xt_lattice_get_info, xt_lattice_s_table,
    xt_lattice_pack_host, xt_particles_init_derived, xt_track, xt_track_ex, xt_track_static, XT_TRACK_STATIC_MAX_PARTICLES, xt_track_host, xt_track_workspace_bytes,
    xt_survival_histogram, xt_twiss4d, xt_twiss4d_chrom, xt_twiss4d_line, xt_twiss4d_normal_form, xt_twiss6d, xt_twiss6d_normal_form, xt_twiss6d_line, xt_refine_loss_location, xt_lattice_set_knobs, xt_track_knobs, xt_fp64_fma_peak, xt_fp64_fma_peak_sweep, xt_fp64_fma_probe, xt_launch_count, xt_build_info,
)
from ._build import build  # noqa: F401
