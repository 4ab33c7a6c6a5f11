"""paper_2412_18553_b200 — B200-native fragment-projected DF-MP2 for SIE embedding clusters.

The product is libsie_dfmp2.so (hand-written sm_100a CUDA behind the C ABI of include/sie_dfmp2.h);
this package is its thin Python binding.  Nothing here computes on the CPU and nothing imports oracle/.
"""
from .binding import (  # noqa: F401
    SIE_FLAG_HOST_IO,
    SIE_FLAG_PROFILE,
    SIE_FLAG_RDM_OCC,
    SIE_FLAG_RDM_VIR,
    SIE_FLAG_REFERENCE,
    SIE_FLAG_STAGE_FULL,
    SIE_FLAG_VALIDATE,
    CanonicalSolver,
    ClusterSolver,
    SieError,
    alloc_workspace,
    launch_count,
    sie_dfmp2_batch,
    sie_dfmp2_batch_query,
    sie_dfmp2_destroy,
    sie_dfmp2_energy,
    sie_dfmp2_energy_lowrank,
    sie_dfmp2_energy_noalloc,
    sie_dfmp2_noalloc_bytes,
    sie_dfmp2_noalloc_capacity,
    sie_dfmp2_rdm_occ,
    sie_dfmp2_rdm_vir,
    sie_dfmp2_plan,
    sie_dfmp2_plan_info,
    sie_dfmp2_plan_reset,
    sie_dfmp2_plan_timing,
    sie_dfmp2_batch_timing,
    sie_dfmp2_probe_fp64,
    sie_dfmp2_transform,
)
