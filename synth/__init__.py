"""Seeded synthetic EXL-50U-shaped inputs.

The one module both the oracle-side tests and the CUDA-side harness import.  It holds none of
the method's arithmetic (no Delta* solve, no search, no fit of basis coefficients, no Picard
loop): it tabulates Green's functions with scipy.special (the offline precompute of
PAPER.md:65-79, which is an INPUT of ptefit_create), lays out a device, and draws per-slice
measurement vectors b and coil currents I_C from analytic D-shaped current distributions.
It imports neither ``oracle`` nor ``paper_2601_12378_b200``.
"""
from .device import CONFIGS, make_device, filament_psi, filament_b   # noqa: F401
from .slices import make_slices                                       # noqa: F401
