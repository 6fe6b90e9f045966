"""B200-native all-pairs softened gravity (Hamada & Iitaka, arXiv astro-ph/0703100), sm_100a only.

The product is ``libnbody_b200.so`` (C ABI, ``include/nbody_b200.h``); this package is the thin
Python binding over it (argument marshalling only) plus the seeded workload generators.
"""
from .binding import (  # noqa: F401
    NBError,
    cunbody_force,
    cunbody_force_jerk_pot,
    cunbody_lennard_jones,
    force,
    force_batched,
    force_eps_i,
    force_host,
    force_jerk,
    force_jerk_host,
    force_packed,
    hermite4,
    hermite4_block_step,
    block_schedule,
    block_step_size,
    last_launch_count,
    leapfrog_kdk,
    pack_j,
    lib,
    plan_query,
    plan_query_jerk,
    plan_query_small,
    debug_set,
    debug_plan_exhaustive,
    debug_plans_computed,
    release_stream,
    profile_enable,
    profile_read,
    release_workspace,
    status_string,
    version,
)
