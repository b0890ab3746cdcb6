"""fp64 CPU oracle of the LASER confidence probe — TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs of
``bench.py`` may import this package.  It shares no code with ``paper_2606_31580_b200`` and never
imports it.  The arithmetic lives in ``laser_oracle.c`` (plain C, IEEE double); this file only
builds that translation unit with gcc and marshals numpy arrays through ctypes.

Citations are to /root/reference/PAPER.md (line numbers) — see the header of laser_oracle.c.
"""
from .binding import (  # noqa: F401
    TauParams, BudgetParams, build, num_threads, row_stats, row_stats_range, merge, aggregate,
    token_prob, SimPolicy, sim_queue, sim_summary,
    tau, tau_scalar, tau_unclamped, exit_mask, probe, ema, budget, f_diff, f_load, ProbeResult,
)
