"""ORACLE -- test infrastructure, NOT product code.

A plain, slow float64 CPU implementation of the ZDA zone solve (arxiv
2501.07979), written from the paper before any CUDA kernel
and sharing no code with ``paper_2501_07979_b200``.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import it.
"""
from .zone import OracleZone, cfl_limit, lens_focal_objective, cpml_profile, radial_coefficients  # noqa: F401
