"""CPU float64 oracle for the SP2 / DNN-SP2 density-matrix path of arXiv 2107.02737.

TEST INFRASTRUCTURE ONLY.  Nothing under ``paper_2107_02737_b200/`` (the CUDA
product path) imports, links or executes this package, and this package imports
nothing from the product.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may call it.

See ``oracle/sp2_oracle.py`` for the functions, each citing the PAPER.md passage
it follows, and ``DESIGN.md`` ("Readings of the paper") for every point where
the paper is silent and a reading had to be chosen.
"""
from .sp2_oracle import (  # noqa: F401
    gershgorin_bounds,
    lanczos_bounds,
    power_trace_bounds,
    rescale_to_unit_interval,
    sp2_stop,
    sp2_density,
    sp2_response_batch,
    sp2_refine_layers,
    congruence,
    density_eigh,
    density_from_eigenpairs,
    response_closed_form,
    response_closed_form_sampled,
    response_finite_difference,
    sp2_spectrum_simulator,
)
