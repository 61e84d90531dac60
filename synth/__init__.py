"""Seeded synthetic inputs for the gridder (arrays, visibilities, weights, kernel tables).

This package only *makes inputs*.  It holds none of the gridding method's arithmetic
(no uvw->cell mapping, no convolution, no binning) and imports neither ``oracle`` nor
``paper_1003_5575_b200``; both of those are fed the same bytes produced here.
The recipe is stated in DESIGN.md ("Input recipe") and follows SURVEY.md section 8(d).
"""
from .workloads import CONFIG_IDS, Workload, config_shape, make_workload  # noqa: F401
from .kernels import spheroidal_1d, spheroidal_table, wplane_tables  # noqa: F401
