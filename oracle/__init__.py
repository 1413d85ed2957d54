"""CPU oracle for the qsGW correlation self-energy build -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product package
``paper_2210_17093_b200`` never does, and this package never imports the product.
"""
from .qsgw_oracle import (  # noqa: F401
    build_library, num_threads, set_num_threads, D, pole_weights, residues, sigma, sigma_diag, ao_to_mo, mp2_direct, mp2, casida_matrix, casida_z, casida,
)
