"""CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference`
legs may import this package.  It shares nothing with paper_2606_17971_b200/.
"""
from .oracle import (  # noqa: F401
    Oracle,
    OracleOptions,
    build_oracle,
    reference_eigs,
    reference_eigs_scaled,
    sine_reference,
    spacetime_reference,
    prolong_p1,
    prolonged_reference,
    transient_reference,
    deflated_spectrum,
    JACOBI_CG,
    REFDEF,
    ZEROEXT,
    INIT_PAPER,
    INIT_ALL_ACTIVE,
    INIT_ALL_INACTIVE,
    INIT_GIVEN,
)
