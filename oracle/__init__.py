"""CPU oracle for the twisted-mass Wilson hot path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this package.  The product path
(``paper_1209_5942_b200``) never does, and this package never imports it.

The arithmetic lives in ``lqcd_oracle.cpp`` and ``gauge_oracle.cpp`` (plain C++17, std::complex<double>);
this module only compiles it with g++ and marshals numpy arrays through ctypes.
Every function cites the passage of PAPER.md it follows in the .cpp file.
"""
from .oracle import (  # noqa: F401
    build,
    gamma,
    m_full,
    dslash_eo,
    dslash_eo_sites,
    mhat,
    mhat_sites,
    mdagm,
    cg_mdagm,
    bicgstab_mhat,
    fermion_force,
    fermion_force_links,
    force_fields,
    force_tm,
    num_threads,
    set_num_threads,
    plaquette,
    staple,
    update_links,
    gauge_subsweep,
    gauge_sweep,
    kp_samples,
)
