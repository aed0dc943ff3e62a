"""B200-native ensemble CN/RK3 DNS step of arXiv 2306.12739 (plane Couette / constant-mass-flux Poiseuille).

The compute path is the C-ABI library `libdns_b200.so` (include/dns.h, csrc/*.cu, sm_100a); `binding` is a
thin ctypes wrapper with the same names.  `inputs` holds the seeded synthetic-input generators only.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding"]
