"""TEST INFRASTRUCTURE ONLY -- the FP64 CPU oracle of the nuclear-pasta MD hot path.

Thin ctypes/numpy marshalling over ``pasta_oracle.c`` (which holds all the arithmetic and the
citations into PAPER.md).  Nothing under ``paper_1412_8502_b200/`` imports this package, and this
package imports nothing from there.  Allowed callers: ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs.
"""
from .pasta_oracle import (  # noqa: F401
    Params,
    build,
    cell_coords,
    cells,
    clusters,
    clusters_cells,
    clusters_mst,
    composition,
    expand,
    forces,
    forces_cells,
    kinetic,
    ncell,
    num_threads,
    pair,
    set_num_threads,
    step,
    step_linear,
    wrap,
)
