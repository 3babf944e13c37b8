"""BASELINE.json configs C1, C3, C4, C5 assembled from the seeded generators.

Input data only: a workload is (HU grid, voxel size, HU->material bins, spot list, history count, seed).
"""
from __future__ import annotations

from .materials import make_materials_c1, make_materials_24
from .phantoms import phantom_c1, phantom_c3, phantom_c4, phantom_c5
from .plans import plan_single_spot, plan_c4, plan_c5

_CACHE = {}


def workload(name: str):
    """name: c1 | c3_70 | c3_150 | c3_230 | c4 | c5  ->  dict(hu, vox, materials, spots, n_histories, seed, label)."""
    if name in _CACHE:
        return _CACHE[name]
    if name == "c1":
        hu, vox = phantom_c1()
        w = dict(hu=hu, vox=vox, materials=make_materials_c1(), spots=plan_single_spot((5.0, 5.0, 0.0), 150.0, 0.3),
                 n_histories=10_000, seed=1,
                 label="C1 water 50x50x100 @2mm, 150 MeV pencil beam sigma 3 mm, 1e4 histories")
    elif name.startswith("c3_"):
        e = float(name.split("_")[1])
        hu, vox = phantom_c3()
        w = dict(hu=hu, vox=vox, materials=make_materials_24(), spots=plan_single_spot((10.0, 10.0, 0.0), e, 0.4),
                 n_histories=1_000_000, seed={70.0: 31, 150.0: 32, 230.0: 33}[e],
                 label=f"C3 slab 200x200x300 @1mm (water/bone/lung/Ti), {e:.0f} MeV sigma 4 mm, 1e6 histories")
    elif name == "c4":
        hu, vox, targets = phantom_c4()
        w = dict(hu=hu, vox=vox, materials=make_materials_24(), spots=plan_c4(hu, vox, targets),
                 n_histories=10_000_000, seed=4,
                 label="C4 synthetic head-and-neck CT 256x256x120 @1x1x2.5mm, 3 fields, 70-200 MeV, 1e7 histories")
    elif name == "c5":
        hu, vox, targets = phantom_c5()
        w = dict(hu=hu, vox=vox, materials=make_materials_24(), spots=plan_c5(hu, vox, targets),
                 n_histories=100_000_000, seed=5,
                 label="C5 synthetic pelvis CT 512x512x200 @1x1x2mm with Ti implants, 2 fields, 100-230 MeV, 1e8 histories")
    else:
        raise ValueError(f"unknown workload {name!r}")
    w["name"] = name
    w["n_spots"] = int(w["spots"].shape[0])
    _CACHE[name] = w
    return w
