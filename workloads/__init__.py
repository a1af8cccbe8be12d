"""Seeded synthetic workloads shaped like the SL1M paper's (arXiv:1310.2078) test problems.

This package holds ONLY input generation (geometry, skies, gain tables, noise draws).  It
contains none of the method's arithmetic: no matrix entry, no operator apply, no solver.  Both
the fp64 oracle (`oracle/`) and the CUDA path (`paper_1310_2078_b200/`) consume these arrays;
neither imports the other.
"""
from .configs import CONFIG_IDS, Workload, make_workload, fista_lambda  # noqa: F401
