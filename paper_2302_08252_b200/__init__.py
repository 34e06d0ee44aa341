"""B200-native AdePT transport step (arXiv 2302.08252 hot path).

The product is the C-ABI library `libadept_b200.so` (include/adept.h); this package is its thin
ctypes binding.  There is no CPU fallback: importing `binding` without the built library raises.
"""
from .binding import (ADEPT_AOS, ADEPT_AOSOA32, ADEPT_AOSOA64, ADEPT_DENSE_DOUBLE, ADEPT_HC16, ADEPT_SOA, ADEPT_SOA16, ADEPT_SPARSE_SINGLE,  # noqa: F401
                      FIELD_NAMES, LAYOUTS, SCHEMES, AdeptError, Context, dev_math, field_offset, lib, step_static)
