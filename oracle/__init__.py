"""float64 CPU oracle for the near-field direct sum -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the product
package ``paper_2110_11398_b200`` and shares no code with it.  See ``nf_oracle.c``
for the definition it writes out and the PAPER.md passages it follows.
"""
from .nf_oracle import (  # noqa: F401
    build,
    kernel,
    bin_particles,
    accel,
    accel_mass,
    density,
    force_scale,
    kick,
    cell_max_accel,
    interactions,
    num_threads,
    OracleError,
)
