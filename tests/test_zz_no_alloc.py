"""pmc_gamma_index_static: the gamma index for callers that may not allocate device memory.

Who needs it: a dose-comparison loop that runs beside a framework whose memory pool already owns the whole GPU (a
cudaMalloc fails there), a loop with a latency budget (cudaMalloc / cudaFree may wait for everything else on the device),
a service that allows no allocation after start-up.  pmc_gamma_index gets its working memory from cudaMalloc or the
context's allocator; this entry point keeps it in one fixed array inside libpmc (8192 search offsets at most) and must
give the same gamma map and pass rate.

What is checked: against pmc_gamma_index on the same inputs, within the tolerance of test_gamma_index.py, on two calls in
a row - the second with a smaller grid, a shorter offset list and a lower maximum, so that anything the first call left
in the shared array (offsets, counts, the maximum) would show; that the context's allocator is never asked for memory;
that a search sphere beyond the fixed size is refused with PMC_E_CAPACITY and the output is left alone.

The file sorts last (pytest --collect-only) on purpose: `pytest -x` stops at the first failure, so a failure here hides
no other test.  It passes alone in a fresh process (the first call then does the one-time address look-up) and after
the rest of the suite."""
import numpy as np
import pytest


def _fields(shape, seed):
    rng = np.random.default_rng(seed)
    z, y, x = np.meshgrid(*(np.arange(n) for n in shape), indexing="ij")
    ref = np.exp(-((x - shape[2] / 2) ** 2 / 200 + (y - shape[1] / 2) ** 2 / 80 + (z - shape[0] / 2) ** 2 / 50))
    ev = np.roll(ref, 1, axis=2) * (1 + 0.02 * rng.standard_normal(shape))
    return ref.astype(np.float32), ev.astype(np.float32)


@pytest.mark.gpu
def test_gamma_index_static_matches_allocating_path_twice_in_a_row():
    import torch
    from paper_1409_8336_b200 import Pmc
    pm_ref = Pmc(0)                                  # existing path: scratch from the context's allocator
    pm = Pmc(0)                                      # the context under test: count what it asks its allocator for
    asked = []
    real_alloc = torch.cuda.caching_allocator_alloc
    # first call: 37 x 45 x 70 voxels of 1 x 1 x 2.5 mm, 2 %/2 mm, search 6 mm (381 offsets), maximum 1;
    # second call: smaller grid of 2 mm voxels, search 4 mm (33 offsets, other values), maximum 0.25, no threshold
    cases = [((37, 45, 70), (0.1, 0.1, 0.25), 0.02, 0.2, 0.1, 1.0, 0.6),
             ((20, 33, 33), (0.2, 0.2, 0.2), 0.02, 0.2, 0.0, 0.25, 0.0)]
    try:
        for shape, vox, dd, dta, low, scale, search in cases:
            ref, ev = _fields(shape, 11)
            ref_d, ev_d = torch.as_tensor(ref * scale, device="cuda"), torch.as_tensor(ev * scale, device="cuda")
            g0, rate0 = pm_ref.gamma_index(ref_d, ev_d, vox, dd, dta, low, search)
            out = torch.full_like(ref_d, 7.0)
            torch.cuda.caching_allocator_alloc = lambda *a, **k: (asked.append(a[0]), real_alloc(*a, **k))[1]
            g1, rate1 = pm.gamma_index_static(ref_d, ev_d, vox, dd, dta, low, search, out=out)
            torch.cuda.caching_allocator_alloc = real_alloc
            assert g1 is out and asked == []                                    # nothing came from the allocator
            g0, g1 = g0.cpu().numpy().astype(np.float64), g1.cpu().numpy().astype(np.float64)
            assert np.array_equal(g0 < 0, g1 < 0)                               # same evaluated set
            m = g0 >= 0
            assert m.sum() > 1000
            assert np.max(np.abs(g1[m] - g0[m])) < 2e-4 * max(1.0, g0[m].max())
            assert abs(rate1 - rate0) <= 2.0 / m.sum()
            assert 0.0 < rate0 < 1.0                                            # the case discriminates
    finally:
        torch.cuda.caching_allocator_alloc = real_alloc
    pm.close(); pm_ref.close()


@pytest.mark.gpu
def test_gamma_index_static_refuses_a_search_sphere_beyond_its_scratch():
    import torch
    from paper_1409_8336_b200 import Pmc, PmcError
    pm = Pmc(0)
    ref = torch.ones((4, 6, 8), device="cuda")
    out = torch.full_like(ref, 7.0)
    with pytest.raises(PmcError) as e:              # radius 1.3 cm of 1 mm voxels: 9171 offsets > 8192
        pm.gamma_index_static(ref, ref, (0.1, 0.1, 0.1), 0.02, 0.2, 0.1, search_cm=1.3, out=out)
    assert e.value.code == -3 and "8192" in str(e.value)                       # PMC_E_CAPACITY, names the limit
    assert float(out.min()) == 7.0 and float(out.max()) == 7.0                 # nothing was written
    g, rate = pm.gamma_index_static(ref, ref, (0.1, 0.1, 0.1), 0.02, 0.2, 0.1, search_cm=1.2, out=out)   # 7153: fits
    assert float(g.abs().max()) == 0.0 and rate == 1.0
    g0, _ = pm.gamma_index(ref, ref * 1.03, (0.1, 0.1, 0.1), 0.02, 0.2, 0.1, search_cm=1.2)
    g1, _ = pm.gamma_index_static(ref, ref * 1.03, (0.1, 0.1, 0.1), 0.02, 0.2, 0.1, search_cm=1.2, out=out)
    assert torch.allclose(g0, g1, atol=1e-5) and abs(float(g1[0, 0, 0]) - 1.5) < 1e-5
    pm.close()
