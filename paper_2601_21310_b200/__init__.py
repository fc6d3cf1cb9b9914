"""paper_2601_21310_b200 — thin Python binding over the detham C ABI (include/detham.h).

Argument marshalling only: every step of the hot path (heat-bath lists, excitation enumeration, Slater-Condon
elements, CSR H_SS, SpMV/energy, PT2 hash accumulation and reduction) runs in the CUDA kernels of libdetham.so.
PyTorch is used for device memory and streams.  There is no CPU fallback: a missing library or device raises.
"""
from .binding import (Detham, DethamError, load_library, use_checked_library, create, energy_static, ENERGY_STATIC_MAX_ROWS, SYMBOLS, STATUS)  # noqa: F401
