"""Float64 CPU oracle for the plasma-line spectral-integration hot path.

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.
It shares nothing with ``paper_2311_18737_b200`` (the CUDA path) and neither imports
the other.  See ``oracle/plspec_oracle.c`` for the arithmetic and its citations
(Eq. 8).
"""
from .profile_oracle import mean_spectrum, profile  # noqa: F401
from .plspec_oracle import (  # noqa: F401
    CF32,
    SC16,
    build,
    fft,
    max_threads,
    spectra,
)
