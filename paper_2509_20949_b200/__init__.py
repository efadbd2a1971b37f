"""B200-native SMC-X hot path (arxiv 2509.20949): thin Python binding over the C-ABI library.

Every step of the hot path runs in the CUDA kernels behind ``include/smcx.h``; this package only
marshals arguments.  PyTorch supplies device memory (the workspace tensor) and the CUDA stream.
There is no CPU fallback: importing works anywhere, but creating a lattice needs ``libsmcx.so``
and a CUDA device and raises otherwise.
"""
from .binding import (  # noqa: F401
    BCC, FCC,
    STORAGE_AUTO, STORAGE_2BIT, STORAGE_4BIT, STORAGE_U8,
    KERNEL_AUTO, KERNEL_WARP_PER_CELL, KERNEL_THREAD_PER_CELL, KERNEL_THREAD_PERSISTENT, KERNEL_GROUP_PER_CELL,
    KERNEL_FCC_THREAD, KERNEL_LOCAL_WARP, KERNEL_BCC4_THREAD, MODEL_EPI, MODEL_LOCAL,
    SmcxError, Lattice, Ensemble, Domain, DomainGroup, load_library, library_path, exported_symbols,
    domain_partition, domain_plan_messages, sro_from_counts, pair_counts_static, STATIC_PAIR_COUNTS_MAX,
)
