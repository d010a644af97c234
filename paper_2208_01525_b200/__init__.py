"""paper_2208_01525_b200 -- B200-native U(1)xU(1) lattice evolution (arXiv:2208.01525 hot path).

The product is libu1u1.so (csrc/, C ABI in include/u1u1.h); this package is its thin binding."""
from .binding import Params, U1U1Error, DIAG_SLOTS, load, state_bytes, scratch_bytes  # noqa: F401
from .lattice import Lattice, Slab, gauss_violation_static  # noqa: F401
