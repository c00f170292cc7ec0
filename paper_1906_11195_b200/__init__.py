"""B200-native multispin Monte Carlo for mean-field spin glasses (arXiv:1906.11195).

Thin Python binding over the C-ABI of include/sg.h (libsg.so).  The binding marshals
arguments only: every step of the path runs in the library's CUDA kernels.
"""
from .binding import (  # noqa: F401
    SG_MODEL_RRBG,
    SG_MODEL_RRG,
    SG_MODEL_SK,
    SG_MODEL_VB,
    SGError,
    Sim,
    kernel_launches,
    load_library,
    sg_correlation,
    sg_create,
    sg_create_opt,
    sg_destroy,
    sg_energy,
    sg_snapshot,
    sg_sweep,
)
from . import workloads  # noqa: F401
