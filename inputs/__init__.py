"""Seeded, synthetic input generators shared by the oracle and the CUDA path.

This package holds INPUT DATA only (physics tables, HU->material tables, CT
phantoms, spot plans).  None of the transport method's arithmetic lives here:
the paper itself treats these as pre-generated inputs (dE/dx and range tables,
f_m(HU), radiation lengths, nuclear cross-section tables "obtained from
Geant4.9.6p2").  Geant4 is not available, so the
tables are generated from closed formulas instead.
Both `oracle/` and `paper_1409_8336_b200/` consume the same bytes, so table
content never enters the parity comparison.
"""
from .physics_tables import make_physics_tables, ELEMENTS  # noqa: F401
from .materials import make_materials_c1, make_materials_24  # noqa: F401
from .phantoms import phantom_c1, phantom_c3, phantom_c4, phantom_c5  # noqa: F401
from .plans import plan_single_spot, plan_c4, plan_c5  # noqa: F401
from .workloads import workload  # noqa: F401
