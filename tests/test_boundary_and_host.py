"""CPU-side tests (`-m "not gpu"`): the C-ABI library loads and exports every symbol include/pmc.h declares,
the host plumbing (history sharding over ranks, workload generators, parity statistics) behaves.
No compute call is made on the library here (there is no GPU and no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import inputs
import paper_1409_8336_b200 as pkg
from paper_1409_8336_b200.sharding import shard_histories, weak_shard, combine_dose
import parity

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "pmc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pmc_[a-z0-9_]+)\s*\(", src)))


def test_header_and_binding_agree():
    assert _declared_symbols() == sorted(pkg.EXPORTS)
    for name in ("pmc_load_ct", "pmc_set_hu_materials", "pmc_load_physics_tables", "pmc_simulate", "pmc_nonelastic"):
        assert name in pkg.EXPORTS            # the five calls of north_star


def test_library_loads_and_exports_every_declared_symbol():
    pkg.build()
    lib = pkg.load_library()
    for name in _declared_symbols():
        assert getattr(lib, name) is not None


def test_no_cpu_fallback():
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    lib = pkg.load_library()
    ctx = ctypes.c_void_p()
    assert lib.pmc_create(ctypes.byref(ctx), 0, None) == -4          # PMC_E_CUDA
    assert not ctx
    with pytest.raises(RuntimeError):
        pkg.Pmc(0)


def test_struct_layouts_match_header():
    from paper_1409_8336_b200 import binding as b
    assert ctypes.sizeof(b.HuBin) == 4 + 4 + 8 * 2 + 8 * 8 + 8 + 8 + 8      # table_id padded to 8
    assert b.SECONDARY_DTYPE.itemsize == 24
    assert inputs.plan_single_spot((0, 0, 0), 100.0, 0.3).shape == (1, 13)     # pmc_spot = 13 doubles


# ------------------------------------------------------------------ sharding
def test_shard_histories_partition():
    for n, world in [(10, 3), (0, 2), (7, 7), (10_000_000, 8), (5, 8)]:
        parts = [shard_histories(n, r, world) for r in range(world)]
        assert parts[0][0] == 0 and sum(c for _, c in parts) == n
        for (o0, c0), (o1, _) in zip(parts[:-1], parts[1:]):
            assert o0 + c0 == o1
        assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
    assert weak_shard(1000, 3) == (3000, 1000)
    with pytest.raises(ValueError):
        shard_histories(10, 2, 2)


def _combine_worker(rank, world, port, tmp):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    g = torch.Generator().manual_seed(100 + rank)
    n_local = [3000, 1000][rank]
    dose = torch.rand(4, 5, 6, generator=g)
    sigma = 0.1 * torch.rand(4, 5, 6, generator=g)
    torch.save((dose.clone(), sigma.clone(), n_local), os.path.join(tmp, f"in{rank}.pt"))
    calls = []
    real = dist.all_reduce
    dist.all_reduce = lambda *a, **k: (calls.append(1), real(*a, **k))[1]      # ONE all-reduce
    d, s, n = combine_dose(dose, sigma, n_local)
    dist.all_reduce = real
    torch.save((d, s, n, len(calls)), os.path.join(tmp, f"out{rank}.pt"))
    dist.destroy_process_group()


def test_combine_dose_gloo_world2(tmp_path):
    port = 29500 + os.getpid() % 2000
    mp.spawn(_combine_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    ins = [torch.load(tmp_path / f"in{r}.pt") for r in range(2)]
    outs = [torch.load(tmp_path / f"out{r}.pt") for r in range(2)]
    n = sum(i[2] for i in ins)
    d_ref = sum(i[0].double() * i[2] for i in ins) / n
    s_ref = torch.sqrt(sum((i[1].double() * i[2] / n) ** 2 for i in ins))
    for d, s, nn, n_calls in outs:
        assert nn == n and n_calls == 1
        assert torch.allclose(d.double(), d_ref, rtol=1e-6, atol=1e-9)
        assert torch.allclose(s.double(), s_ref, rtol=1e-6, atol=1e-9)


# ------------------------------------------------------------------ input recipe
def test_workloads_have_the_configured_shapes():
    w = inputs.workload("c1")
    assert w["hu"].shape == (100, 50, 50) and w["vox"] == (0.2, 0.2, 0.2) and w["n_histories"] == 10_000
    assert np.all(w["hu"] == 0) and w["spots"][0, 6] == 150.0 and w["spots"][0, 8] == 0.3
    w = inputs.workload("c3_150")
    assert w["hu"].shape == (300, 200, 200) and len(w["materials"]) == 24
    assert w["hu"][55, 0, 0] == 1200 and w["hu"][100, 0, 0] == -700 and w["hu"][150, 100, 100] == 3071
    w = inputs.workload("c4")
    assert w["hu"].shape == (120, 256, 256) and w["vox"] == (0.1, 0.1, 0.25) and w["n_histories"] == 10_000_000
    e = w["spots"][:, 6]
    assert 1500 <= w["n_spots"] <= 2600 and e.min() >= 70.0 and e.max() <= 200.0 and e.max() > 150.0
    assert w["hu"].min() == -1000 and w["hu"].max() >= 2000
    d = w["spots"][:, 3:6]
    assert len({tuple(np.round(x, 6)) for x in d}) == 3                  # three fields
    hu2, _, _ = inputs.phantom_c4()
    assert np.array_equal(hu2, w["hu"])                                  # seeded: reproducible


def test_materials_table_is_contiguous_and_normalised():
    for mats in (inputs.make_materials_c1(), inputs.make_materials_24()):
        for a, b in zip(mats[:-1], mats[1:]):
            assert a["hu_hi"] == b["hu_lo"]
        for m in mats:
            assert abs(np.sum(m["w"]) - 1) < 1e-12 and m["rho_lo"] > 0 and m["x0_gcm2"] > 0


# ------------------------------------------------------------------ parity statistics helpers
def test_distal_depth_on_an_analytic_curve():
    z = (np.arange(200) + 0.5) * 0.1
    dd = np.where(z < 10, 1.0 + 0.1 * z, np.clip(2.0 - (z - 10.0) / 0.5, 0, None))     # linear fall 10 -> 11 cm
    r80, fall = parity.r80_and_falloff(dd, 0.1)
    peak = 1.0 + 0.1 * 9.95                       # the curve is 2 - (z - 10)/0.5 beyond the peak
    assert abs(r80 - (10.0 + 0.5 * (2.0 - 0.8 * peak))) < 1e-9
    assert abs(fall - 0.5 * 0.6 * peak) < 1e-9


def test_zscore_pass_rate_under_the_null():
    rng = np.random.default_rng(0)
    truth = np.linspace(1, 10, 20000)
    a = truth + rng.normal(0, 0.1, truth.size); b = truth + rng.normal(0, 0.1, truth.size)
    frac, mean, rms, n = parity.zscore_pass(a, np.full_like(a, 0.1), b, np.full_like(b, 0.1))
    assert n > 15000 and frac > 0.995 and abs(mean) < 0.05 and abs(rms - 1) < 0.05
    frac2, *_ = parity.zscore_pass(a + 0.5, np.full_like(a, 0.1), b, np.full_like(b, 0.1))
    assert frac2 < 0.5
