"""CPU oracle for the plane-wave H.Psi / Chebyshev-filter / Gram hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It does not import, link or call anything from paper_2604_11139_b200 (the CUDA path), and the CUDA path
never imports it.  See oracle/pw_oracle.c for the definitions and citations, DESIGN.md section 2 for the pins.
"""
from .pw_oracle import (apply_h, build, cheb_filter, dft1d, dft3d, fft1d, gram, kinetic, n_threads,  # noqa: F401
                        TERM_KIN, TERM_LOC, TERM_NL, TERM_ALL)
from .dense import dense_h  # noqa: F401
from . import density_oracle as density_oracle  # noqa: F401   (density, band sharding)
from . import lobpcg_oracle as lobpcg_oracle  # noqa: F401   (LOBPCG block solve)
from . import paw_oracle as paw  # noqa: F401   (PAW-style generalised problem)
from . import rr_oracle as rr  # noqa: F401   (Rayleigh-Ritz companion steps)
