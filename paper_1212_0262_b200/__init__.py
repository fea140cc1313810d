"""B200-native (sm_100a) hot path of arXiv 1212.0262: long-range N-body molecular dynamics
(HMF, Ring, 2D self-gravity) with a 4th-order symplectic integrator, behind the C ABI of
``include/lrmd.h``.  ``lrmd`` is the binding; ``inputs`` the seeded synthetic workloads."""
from . import inputs, lrmd  # noqa: F401
from .lrmd import GRAV2D, HMF, RING, Context, LrmdError  # noqa: F401
