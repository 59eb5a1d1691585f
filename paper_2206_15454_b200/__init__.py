"""B200-native fused D3Q19 LES + forest-canopy lattice Boltzmann step (arxiv 2206.15454).

The product is the C-ABI CUDA library `liblbm_b200.so` (include/lbm.h); this package is its
thin Python binding.  It never imports `oracle/`.
"""
from .binding import (  # noqa: F401
    Lbm, LbmError, bc_flags, workspace_bytes, lad_profile, lad_from_spec, mix64, lib, SYMBOLS,
    wall_friction_velocity, forest_friction_velocity, stats_normalise, wall_units, stats_from_raw,
    forest_code, forest_codes_from_spec, lad_eq14, sgs_van_driest, sgs_mean_shear, plane_stats_static, STATIC_SCRATCH_BYTES,
    BOTTOM_WALL, BOTTOM_PERIODIC, TOP_WALL, TOP_FREE_SLIP, TOP_PERIODIC, TOP_FORCED_EQ, DRAG_VECTOR, SOLID_MASK, STORAGE_AA, STORAGE_AAX, Z_HALO,
    INIT_POWER_LAW, INIT_PARABOLA, INIT_REST, NSTAT,
    LBM_OK, LBM_EINVAL, LBM_ENOMEM, LBM_ESTATE, LBM_ECUDA, LBM_EDIVERGED,
)
