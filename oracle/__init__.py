"""oracle — TEST INFRASTRUCTURE, NOT PRODUCT.

ctypes/numpy front end of ``qw_oracle.cpp``: the plain double-precision CPU definition of
the coined-quantum-walk step ``U = S (I (x) C)`` (PAPER.md:42 eq. 2, :80 eq. 7).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; it imports nothing from
``paper_1003_3779_b200`` and the product never imports it.
"""
from .oracle import (  # noqa: F401
    build,
    dense_unitary,
    moments,
    philox4x32_10,
    probabilities,
    probabilities_mean,
    rbl_mask,
    step,
    step_inverse,
    step_inverse_rbl,
    step_rbl,
)
