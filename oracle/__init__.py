"""TEST INFRASTRUCTURE: the fp64 CPU oracle (oracle/qmc_oracle.c) and its ctypes binding.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It imports nothing from paper_1802_06922_b200.
"""
from .binding import (  # noqa: F401
    build,
    spline_vgl,
    spline_vgl_twist,
    lu_inverse,
    binv_from_A,
    det_ratio,
    sm_update,
    slater_matrix,
    det_kinetic,
    init_walkers,
    sweep,
    wf_sweep,
    max_threads,
    Jastrow,
    b3,
    jastrow_u,
    min_image,
    jastrow_value,
    jastrow_dj,
)
