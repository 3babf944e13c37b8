"""3-D gamma index: pins of the fp64 oracle (`-m "not gpu"`) and parity of the
CUDA kernel behind pmc_gamma_index against it (`-m gpu`, element by element)."""
import numpy as np
import pytest

from oracle.gamma import gamma_index

VOX = (0.1, 0.1, 0.25)


def _brute(ref, ev, vox, dd_frac, dta, low, search):
    """Pure-Python triple loop over every pair of voxels: the definition with nothing vectorised (tiny grids only)."""
    nz, ny, nx = ref.shape
    dmax = ref.max(); dd = dd_frac * dmax
    out = np.full(ref.shape, -1.0)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                if ref[k, j, i] < low * dmax:
                    continue
                best = np.inf
                for kk in range(nz):
                    for jj in range(ny):
                        for ii in range(nx):
                            d2 = ((ii - i) * vox[0]) ** 2 + ((jj - j) * vox[1]) ** 2 + ((kk - k) * vox[2]) ** 2
                            if d2 > search * search * (1 + 1e-12):
                                continue
                            best = min(best, d2 / dta ** 2 + (ev[kk, jj, ii] - ref[k, j, i]) ** 2 / dd ** 2)
                out[k, j, i] = np.sqrt(best)
    return out


def test_gamma_oracle_against_brute_force_tiny():
    rng = np.random.default_rng(1)
    ref = rng.random((4, 5, 6)) + 0.2
    ev = ref * (1 + 0.05 * rng.standard_normal(ref.shape))
    g, _ = gamma_index(ref, ev, VOX, 0.03, 0.2, 0.3, 0.4)
    assert np.allclose(g, _brute(ref, ev, VOX, 0.03, 0.2, 0.3, 0.4), rtol=1e-12, atol=1e-12)


def test_gamma_oracle_closed_forms():
    ref = np.full((6, 12, 12), 2.0)
    # identical doses: gamma = 0, pass rate 1
    g, p = gamma_index(ref, ref, VOX)
    assert np.all(g == 0) and p == 1.0
    # uniform fields differing by delta: no neighbour is closer in dose, gamma = |delta| / dd_frac everywhere
    g, p = gamma_index(ref, ref * 1.03, VOX, dd_frac=0.02)
    assert np.allclose(g, 1.5) and p == 0.0
    g, p = gamma_index(ref, ref * 0.99, VOX, dd_frac=0.02)
    assert np.allclose(g, 0.5) and p == 1.0
    # a step edge displaced by one 1 mm voxel along x, DTA 2 mm: the voxels the edge moved over find their dose one
    # voxel away (gamma = 1 mm / 2 mm = 0.5), all the others at distance 0
    step = np.zeros((4, 8, 16)); step[:, :, 8:] = 1.0
    moved = np.zeros_like(step); moved[:, :, 9:] = 1.0
    g, _ = gamma_index(step, moved, VOX, 0.02, 0.2, 0.0)
    expect = np.zeros_like(step); expect[:, :, 8] = 0.5
    assert np.allclose(g, expect)
    # linear ramp D = a x against itself displaced by s voxels: min over lattice offsets t of
    # sqrt((t h)^2 / DTA^2 + (a (t - s) h)^2 / dD^2), checked in the interior
    a, s, h = 0.05, 1, VOX[0]
    x = np.arange(40) * h
    ramp = np.broadcast_to(1.0 + a * x / h, (3, 3, 40)).copy()
    shifted = np.broadcast_to(1.0 + a * (x / h - s), (3, 3, 40)).copy()
    dd, dta = 0.02 * ramp.max(), 0.2
    expect = min(np.sqrt((t * h) ** 2 / dta ** 2 + (a * (t - s)) ** 2 / dd ** 2) for t in range(-4, 5))
    g, _ = gamma_index(ramp, shifted, VOX, 0.02, dta, 0.0)
    assert np.allclose(g[1, 1, 6:34], expect)
    # below the low-dose threshold: -1
    low = ref.copy(); low[0] = 0.1
    g, _ = gamma_index(low, low, VOX, 0.02, 0.2, 0.1)
    assert np.all(g[0] == -1) and np.all(g[1:] == 0)


@pytest.mark.gpu
@pytest.mark.parametrize("shape,vox,dd,dta", [((37, 45, 70), (0.1, 0.1, 0.25), 0.02, 0.2),
                                              ((20, 33, 33), (0.2, 0.2, 0.2), 0.03, 0.3),
                                              ((5, 7, 130), (0.1, 0.15, 0.3), 0.01, 0.1)])
def test_gamma_kernel_matches_oracle(shape, vox, dd, dta):
    import torch
    from paper_1409_8336_b200 import Pmc
    rng = np.random.default_rng(7)
    z, y, x = np.meshgrid(*(np.arange(n) for n in shape), indexing="ij")
    ref = np.exp(-((x - shape[2] / 2) ** 2 / 200 + (y - shape[1] / 2) ** 2 / 80 + (z - shape[0] / 2) ** 2 / 50))
    ev = np.roll(ref, 1, axis=2) * (1 + 0.02 * rng.standard_normal(shape))
    ref32, ev32 = ref.astype(np.float32), ev.astype(np.float32)
    pm = Pmc(0)
    g, rate = pm.gamma_index(torch.as_tensor(ref32, device="cuda"), torch.as_tensor(ev32, device="cuda"), vox, dd, dta, 0.1)
    go, rate_o = gamma_index(ref32, ev32, vox, dd, dta, 0.1)
    g = g.cpu().numpy().astype(np.float64)
    assert np.array_equal(g < 0, go < 0)                                   # same evaluated set
    m = go >= 0
    assert np.max(np.abs(g[m] - go[m])) < 2e-4 * max(1.0, go[m].max())     # fp32 arithmetic of the same minimum
    assert abs(rate - rate_o) <= 2.0 / m.sum()                              # voxels sitting on gamma = 1 within rounding
    pm.close()


@pytest.mark.gpu
def test_gamma_kernel_edge_cases():
    import torch
    from paper_1409_8336_b200 import Pmc, PmcError
    pm = Pmc(0)
    ref = torch.full((3, 4, 5), 2.0, device="cuda")
    g, rate = pm.gamma_index(ref, ref * 1.03, VOX, 0.02, 0.2, 0.1)
    assert torch.allclose(g, torch.full_like(g, 1.5), atol=1e-5) and rate == 0.0
    g, rate = pm.gamma_index(ref, ref, VOX, 0.02, 0.2, 0.1)
    assert float(g.abs().max()) == 0.0 and rate == 1.0
    zero = torch.zeros((3, 4, 5), device="cuda")
    g, rate = pm.gamma_index(zero, zero, VOX, 0.02, 0.2, 0.1)              # all-zero reference: nothing to evaluate
    assert float(g.max()) == -1.0 and rate == 1.0
    one = torch.ones((1, 1, 1), device="cuda")
    g, rate = pm.gamma_index(one, one * 1.01, VOX, 0.02, 0.2, 0.1)        # single voxel
    assert abs(float(g[0, 0, 0]) - 0.5) < 1e-5
    with pytest.raises(PmcError):
        pm.gamma_index(ref, ref, VOX, 0.0, 0.2, 0.1)
    with pytest.raises(PmcError):
        pm.gamma_index(ref, ref, (0.1, -0.1, 0.1), 0.02, 0.2, 0.1)
    pm.close()
