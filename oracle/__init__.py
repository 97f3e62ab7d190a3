"""float64 CPU oracle for the batched RBM local energy -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The product (paper_2108_03409_b200/) never does, and this package never
imports the product.  See oracle/nqs_oracle.c for what is computed and the citations.
"""
from .oracle import (  # noqa: F401
    build,
    connected,
    forces,
    lncosh,
    local_energy_definition,
    local_energy_fast,
    log_derivatives,
    log_psi,
    mean_variance,
    metropolis,
    num_threads,
    set_num_threads,
)
from .fisher import fisher, fisher_from_derivatives  # noqa: F401,E402
