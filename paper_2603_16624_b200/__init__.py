"""paper_2603_16624_b200 -- Python binding of libecpush, the B200-native (sm_100a, FP64) particle
hot path of the ECsim scheme (arxiv 2603.16624): gather, rotation matrix, push, and deposit of
rho, Jhat and the 27-neighbour mass matrices.

The binding only marshals arguments (ctypes) into the C ABI declared in include/ecpush.h; every
step of the path runs in the CUDA kernels of csrc/.  PyTorch is used for device memory and
streams only.  There is no CPU fallback: if libecpush.so is missing or a call fails, an
exception is raised.
"""
from .binding import (  # noqa: F401
    EcsimError,
    Ecsim,
    lib,
    lib_path,
    declared_symbols,
    VARIANT_ATOMIC,
    VARIANT_FUSED,
    ACC_NONE,
    ACC_ALL,
    ACC_M_ONLY,
    M_27,
    M_14,
    STATIC_MAX_CELLS,
    cell_segments_static,
)
