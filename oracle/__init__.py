"""ORACLE - test infrastructure only.

A plain double-precision CPU statement of the SPD hot path written from
/root/reference/PAPER.md, plus the paper's sensitivity formulae.  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import it; the product package never does.
"""
from . import formulas  # noqa: F401
from .core import (  # noqa: F401
    build,
    cluster_candidates,
    find_candidates,
    num_threads,
    row_stats,
    row_stats_clipped,
    snr_of_width,
    spd_direct,
    spd_direct_sw,
    width_sigma,
    spd_grid,
    spd_grid_iter,
    grid_iterations,
    spd_grid_sw,
    spd_prefix,
)
