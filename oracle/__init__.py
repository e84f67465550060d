"""CPU oracle for two-stage subband dedispersion — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA
package ``paper_2110_12749_b200`` and shares no code with it.
"""
from .oracle import (  # noqa: F401
    build_oracle,
    delay_tables,
    dedisperse,
    geometry,
    points,
    max_threads,
    rfi_prologue,
    search,
)
