"""CPU oracle for the pCT hot path -- TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_1707_05014_b200`` (the CUDA path) and neither imports the other.

The arithmetic lives in ``pct_oracle.c`` (plain C, fp64 definitions + a scalar mirror of the
fp32 rule); this module only builds it with gcc and marshals arguments through ctypes.
"""
from .binding import (  # noqa: F401
    Geometry,
    Histories,
    block_accumulate,
    build,
    carp_iterate,
    drop_iterate,
    get_path_model,
    get_substeps,
    get_walk_mode,
    lib,
    mlp_chi2_f64,
    mlp_matrix_f64,
    num_threads,
    path_f64,
    row_f32,
    rule_log,
    scatter_f,
    set_path_model,
    set_substeps,
    set_walk_mode,
    sigma1_table,
    sigma_f64,
    xyz_to_beam_f32,
    xyz_to_beam_f64,
)
