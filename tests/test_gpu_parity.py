"""GPU parity tests (`-m gpu`): the CUDA path, called through the C-ABI of include/pmc.h, against the fp64 oracle.

Philox is compared bit for bit; table evaluation element by element; everything downstream statistically with
north_star's tolerances (identical Philox streams diverge at fp32-vs-fp64 branch points):
integrated dose 0.5 %, >= 99 % of voxels above 10 % of the maximum within 3 combined sigma, R80 and distal
fall-off 0.2 mm, secondary yields 3 sigma, charge / baryon number exact.
"""
import numpy as np
import pytest
import torch

import inputs
import parity
from oracle import Oracle
from oracle import binding as ob

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pm(tables):
    from paper_1409_8336_b200 import Pmc
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device (there is no CPU fallback)"
    p = Pmc(0)
    p.load_physics_tables(tables)
    yield p
    p.close()


def _setup(pm, tables, mats, hu, vox, **opts):
    """Same tables / materials / CT / options on both sides -> (pm, oracle)."""
    pm.load_physics_tables(tables)
    pm.set_hu_materials(mats)
    pm.load_ct(torch.as_tensor(hu, device="cuda"), vox)
    o = Oracle(tables, mats)
    o.load_ct(hu, vox)
    for k in ("straggling", "mcs", "elastic", "nonelastic"):
        pm.set_option(k, float(opts.get(k, 1)))
        o.set_option(k, float(opts.get(k, 1)))
    return o


# ------------------------------------------------------------------ S0 Philox: bit-exact
def test_philox_bit_exact_against_kat_and_oracle(pm):
    kat = [((0, 0, 0, 0), (0, 0), (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
           ((0xffffffff,) * 4, (0xffffffff,) * 2, (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
           ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0),
            (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1))]
    rng = np.random.default_rng(5)
    rnd = rng.integers(0, 2 ** 32, size=(1000, 6), dtype=np.uint64).astype(np.uint32)
    rows = np.array([list(c) + list(k) for c, k, _ in kat], dtype=np.uint32)
    out = pm.philox4x32_10(np.concatenate([rows, rnd]))
    for i, (_, _, ref) in enumerate(kat):
        assert tuple(int(x) for x in out[i]) == ref
    for i in range(0, 1000, 7):
        r = rnd[i]
        assert [int(x) for x in out[3 + i]] == ob.philox4x32_10([int(x) for x in r[:4]], [int(x) for x in r[4:]])


def test_philox_empty_input(pm):
    assert pm.philox4x32_10(np.zeros((0, 6), dtype=np.uint32)).shape == (0, 4)


# ------------------------------------------------------------------ S4 range tables: element by element
@pytest.mark.parametrize("table", [0, 1, 2])
def test_range_tables_match_oracle(pm, oracle_c1, table):
    # fp32 evaluation of ln R splines: |d ln R| <~ 16 ulp(ln R ~ 5) ~ 1e-5 relative
    e = np.exp(np.linspace(np.log(0.06), np.log(290.0), 4099)).astype(np.float32)          # ragged size
    r_g = pm.range_of_energy(table, e).astype(np.float64)
    r_o = np.array([oracle_c1.range_gcm2(table, float(x)) for x in e])
    assert np.max(np.abs(r_g / r_o - 1)) < 3e-5
    e_back = pm.energy_of_range(table, r_g.astype(np.float32)).astype(np.float64)
    e_o = np.array([oracle_c1.energy_of_range(table, float(x)) for x in r_g])
    assert np.max(np.abs(e_back / e_o - 1)) < 3e-5
    assert np.max(np.abs(e_back / e - 1)) < 1e-4


@pytest.mark.parametrize("mats_name,hu_bin", [("c1", 0), ("c1", 1), ("c1", 2), ("24", 1), ("24", 23)])
def test_step_kernel_table_lookup_matches_oracle(pm, tables, oracle_c1, mats_name, hu_bin):
    # the production look-up of the step kernel (shared-memory tables, knot index from log2 E in one FMA, interleaved
    # knots, MUFU log2 / exp2), element by element.  On top of the 1e-5 of the spline evaluation: the fp32 knot coordinate
    # of up to 255 carries up to ~3e-5 knots (2^-24 of itself and of its two constants), i.e. ~2e-6 of R with
    # d ln R / d knot = 0.06; lg2.approx / ex2.approx add ~2 ulp of ln R ~ 5 and of the result: 4e-5 in all
    mats = inputs.make_materials_c1() if mats_name == "c1" else inputs.make_materials_24()
    pm.load_physics_tables(tables); pm.set_hu_materials(mats)
    table = mats[hu_bin]["table_id"]
    e = np.exp(np.linspace(np.log(0.06), np.log(290.0), 70001)).astype(np.float32)          # several blocks, ragged tail
    r_g = pm.step_range_of_energy(hu_bin, e).astype(np.float64)
    r_o = np.array([oracle_c1.range_gcm2(table, float(x)) for x in e[::17]])
    assert np.max(np.abs(r_g[::17] / r_o - 1)) < 4e-5
    assert np.max(np.abs(r_g / pm.range_of_energy(table, e) - 1)) < 5e-5                    # every element, vs the plain path
    e_back = pm.step_energy_of_range(hu_bin, r_g.astype(np.float32)).astype(np.float64)
    e_o = np.array([oracle_c1.energy_of_range(table, float(x)) for x in r_g[::17]])
    assert np.max(np.abs(e_back[::17] / e_o - 1)) < 4e-5
    assert np.max(np.abs(e_back / e - 1)) < 1e-4
    # clamps of the step kernel: below / above the table the end values come back
    lo_hi = pm.step_range_of_energy(hu_bin, np.array([1e-3, 1e4], dtype=np.float32))
    assert lo_hi[0] == pytest.approx(oracle_c1.range_gcm2(table, 0.05), rel=4e-5)
    assert lo_hi[1] == pytest.approx(oracle_c1.range_gcm2(table, 300.0), rel=4e-5)
    assert pm.step_range_of_energy(hu_bin, np.zeros(0, dtype=np.float32)).shape == (0,)


# ------------------------------------------------------------------ S5 straggling: cumulants and distribution
@pytest.mark.parametrize("e_mev,rho_l", [(230.0, 0.1), (150.0, 0.2), (70.0, 0.2), (30.0, 0.25), (5.0, 0.02), (200.0, 0.0003)])
def test_straggling_distribution(pm, oracle_c1, e_mev, rho_l):
    zoa, n = 0.555087, 400_000
    mean = 0.5 * rho_l * 5.0 + (0.01 if rho_l < 0.001 else 0.0)          # (the 3 um step: keep the loss clear of the clamp at 0)
    g = pm.straggle(e_mev, mean, rho_l, zoa, n, 11).astype(np.float64)
    o = oracle_c1.straggle(e_mev, mean, rho_l, zoa, n, 12)
    sd = o.std()
    assert abs(g.mean() - o.mean()) < 5 * sd / np.sqrt(n) * np.sqrt(2) + 1e-6
    # (sampling error of a variance: sqrt((kurtosis - 1)/n); the 3 um step is Landau-like, kurtosis ~ 1/(3 kappa) = 2000)
    kurt = np.mean((o - o.mean()) ** 4) / o.var() ** 2
    assert abs(g.var() / o.var() - 1) < max(0.03, 4 * np.sqrt(2 * (kurt - 1) / n))
    m3g, m3o = np.mean((g - g.mean()) ** 3), np.mean((o - o.mean()) ** 3)
    if kurt < 100:
        assert abs(m3g - m3o) < 0.15 * abs(m3o) + 0.02 * sd ** 3
    # quantiles of the bulk agree to a small fraction of the width
    q = np.array([0.01, 0.05, 0.25, 0.5, 0.75, 0.95, 0.99])
    assert np.max(np.abs(np.quantile(g, q) - np.quantile(o, q))) < 0.03 * sd


@pytest.mark.parametrize("e_mev,rho_l", [(230.0, 0.1), (150.0, 0.2), (70.0, 0.2), (30.0, 0.25), (200.0, 0.02)])
def test_straggling_against_the_vavilov_distribution_itself(pm, e_mev, rho_l):
    """The CUDA sampler (hard collisions + shifted-gamma soft part, Reading R4) against Vavilov's distribution computed from
    its characteristic function (tests/vavilov_ref.py) - a reference that involves neither the oracle nor any sampling.
    kappa from 0.011 to 5.3; Kolmogorov distance below 0.6 % (4e5 samples resolve 0.3 %; measured 0.1-0.3 %).  Thinner steps
    (xi below a few keV) are outside this comparison: Reading R4 lumps the collisions below 1 keV into a Gaussian of
    variance xi x 1 keV on BOTH sides, which is then wider than Vavilov's own sub-keV structure (0.3 keV - immaterial for the
    dose); there the CUDA sampler is compared with the oracle (test_straggling_distribution, the 3 um case)."""
    from scipy import stats
    from vavilov_ref import vavilov_cdf
    from inputs.physics_tables import M_P, M_E, K_BETHE
    g_ = 1 + e_mev / M_P; b2 = 1 - 1 / g_ ** 2
    tmax = 2 * M_E * b2 * g_ * g_ / (1 + 2 * g_ * M_E / M_P + (M_E / M_P) ** 2)
    xi = 0.5 * K_BETHE * 0.555087 * rho_l / b2
    kappa = xi / tmax
    mean_loss = 8.0 * xi + 2.0 * np.sqrt(xi * tmax) + 0.5
    x = pm.straggle(e_mev, mean_loss, rho_l, 0.555087, 400_000, 123).astype(np.float64)
    y, cdf = vavilov_cdf(kappa, b2)
    d = stats.kstest((x - mean_loss) / tmax, lambda t: np.interp(t, y, cdf)).statistic
    print(f"kappa {kappa:.3g}: Kolmogorov distance to Vavilov {d:.4f}")
    assert d < 0.006, (kappa, d)


# ------------------------------------------------------------------ S10 nuclear elastic (Eq.3) and p-p
@pytest.mark.parametrize("Z,A,t_mev", [(8, 16, 150.0), (20, 40, 100.0), (22, 48, 200.0), (1, 1, 150.0)])
def test_elastic_matches_oracle(pm, oracle_c1, tables, Z, A, t_mev):
    from scipy import stats
    n = 200_000
    g = pm.elastic(Z, A, t_mev, n, 41).astype(np.float64)
    o = oracle_c1.elastic(Z, A, t_mev, n, 42)
    assert stats.ks_2samp(g[:, 0], o[:, 0]).pvalue > 1e-3                  # |t| distribution
    assert stats.ks_2samp(g[:, 3], o[:, 3]).pvalue > 1e-3                  # opening angle
    assert np.allclose(g[:, 1] + g[:, 2], t_mev, atol=2e-4)               # fp32 energy conservation
    m_t = tables["nuclear_mass"][Z, A]
    assert np.allclose(g[:, 2], g[:, 0] * 1e6 / (2 * m_t), rtol=1e-5, atol=1e-6)
    assert abs(g[:, 2].mean() - o[:, 2].mean()) < 5 * o[:, 2].std() * np.sqrt(2 / n)


# ------------------------------------------------------------------ S3-S6 first steps: MCS / hinge / energy moments
@pytest.mark.parametrize("e_mev,max_steps", [(150.0, 1), (70.0, 5), (230.0, 40)])
def test_first_steps_moments_match_oracle(pm, tables, e_mev, max_steps):
    hu, vox = inputs.phantom_c1()
    o = _setup(pm, tables, inputs.make_materials_c1(), hu, vox, elastic=0, nonelastic=0)
    # the pencil starts at a voxel centre: on a voxel face (x = 5.0) the first deflection decides the voxel and the
    # one-step x distribution is one-sided, with the side set by how 5.0/0.2 rounds in fp32 vs fp64
    spot = inputs.plan_single_spot((5.1, 5.1, 0.0), e_mev, 0.0)
    n = 200_000
    # s_max incommensurate with the 2 mm voxel: with the default (0.2 cm = the voxel) every deflected step is a
    # near-tie between s_max and the face, and the depth after k steps depends on fp32-vs-fp64 rounding
    pm.set_option("s_max_wet_cm", 0.07); o.set_option("s_max_wet_cm", 0.07)
    try:
        g = pm.first_steps(spot, n, 5, max_steps).astype(np.float64)
        r = o.first_steps(spot, n, 6, max_steps)
    finally:
        pm.set_option("s_max_wet_cm", 0.2)
    se = np.sqrt(2.0 / n)
    for col, name in [(0, "x"), (1, "y"), (3, "u"), (4, "v")]:
        sg, so = g[:, col].std(), r[:, col].std()
        assert abs(g[:, col].mean() - r[:, col].mean()) < 5 * so * se, name
        assert abs(sg / so - 1) < 0.02, name                               # widths (Highland x 1.07, hinge)
    # angle-displacement covariance of the hinge (Fermi-Eyges)
    cg, co = np.mean((g[:, 0] - 5.1) * g[:, 3]), np.mean((r[:, 0] - 5.1) * r[:, 3])
    assert abs(cg / co - 1) < 0.05
    # depth, energy and path length after max_steps
    for col, name in [(2, "z"), (6, "E"), (7, "path")]:
        so = max(r[:, col].std(), 1e-9)
        assert abs(g[:, col].mean() - r[:, col].mean()) < 5 * so * se + 2e-6 * abs(r[:, col].mean()), name
    assert abs(g[:, 6].std() / r[:, 6].std() - 1) < 0.03                  # straggling width


def test_first_steps_deterministic_limits(pm, tables):
    # all fluctuations off: every history is the same CSDA track; compare element by element (fp32 vs fp64)
    hu, vox = inputs.phantom_c1()
    o = _setup(pm, tables, inputs.make_materials_c1(), hu, vox, straggling=0, mcs=0, elastic=0, nonelastic=0)
    spot = inputs.plan_single_spot((5.0, 5.0, 0.0), 150.0, 0.3)
    g = pm.first_steps(spot, 1000, 5, 30).astype(np.float64)
    r = o.first_steps(spot, 1000, 5, 30)
    assert np.allclose(g[:, 2], r[:, 2], atol=2e-5) and np.allclose(g[:, 7], r[:, 7], atol=2e-5)
    assert np.allclose(g[:, 6], r[:, 6], rtol=2e-5)                       # 30 range-table updates in fp32
    assert np.allclose(g[:, 3:6], [0, 0, 1], atol=1e-7)
    # the draw order of the two sides is free: the spot profile is compared as a distribution
    assert abs(g[:, 0].std() / 0.3 - 1) < 0.1 and abs(r[:, 0].std() / 0.3 - 1) < 0.1


def test_odd_table_and_bin_counts(monkeypatch):
    # 255 energy knots and 3 HU bins, both odd: the step kernel's 8-byte HU table then follows an odd number of 4-byte
    # words in shared memory and has to be aligned by address (it used to fault with "misaligned address")
    from paper_1409_8336_b200 import Pmc
    import inputs.physics_tables as pt
    monkeypatch.setattr(pt, "N_E", 255); monkeypatch.setattr(pt, "N_R", 253)
    t_odd = inputs.make_physics_tables()
    assert t_odd["n_e"] == 255 and t_odd["ln_range"].shape[1] == 255 and len(inputs.make_materials_c1()) == 3
    p = Pmc(0)
    hu, vox = inputs.phantom_c1()
    o = _setup(p, t_odd, inputs.make_materials_c1(), hu, vox, straggling=0, mcs=0, elastic=0, nonelastic=0)
    spot = inputs.plan_single_spot((5.0, 5.0, 0.0), 150.0, 0.3)
    g = p.first_steps(spot, 1000, 5, 30).astype(np.float64)
    r = o.first_steps(spot, 1000, 5, 30)
    # fp32 knot coordinate t = log2(E) c1 - c0 of up to 255 carries up to ~3e-5 knots of rounding (2^-24 of t and of the two
    # constants), i.e. ~1e-6 of E per table look-up with knots 3.4 % apart, of one sign for a given table size: 30 steps of
    # forward + inverse look-up stay below 6e-5 (seen: 4e-7 with 256 knots, 2.3e-5 with 255)
    assert np.allclose(g[:, 2], r[:, 2], atol=2e-5) and np.allclose(g[:, 6], r[:, 6], rtol=6e-5)
    for k in ("straggling", "mcs", "elastic", "nonelastic"):
        p.set_option(k, 1.0)
    dose, _ = p.simulate(spot, 20000, 3)                                   # the production instantiation, full physics
    c = p.counters()
    dd = dose.sum(dim=(1, 2)).cpu().numpy()
    assert 15.2 < (np.argmax(dd) + 0.5) * vox[2] < 15.9 and c["n_nonelastic"] > 0     # Bragg peak of 150 MeV in water
    p.close()


# ------------------------------------------------------------------ S12-S13 non-elastic collisions (config C2)
C2_CASES = [(6, 12), (8, 16), (20, 40), (22, 48)]


@pytest.mark.parametrize("Z,A", C2_CASES)
@pytest.mark.parametrize("ie,e_mev", [(0, 100.0), (1, 200.0)])
def test_nonelastic_c2_yields_spectra_angles(pm, oracle_c1, tables, Z, A, ie, e_mev):
    n = 100_000                                                            # C2: 1e5 events per target and energy
    seed = 2000 + 10 * C2_CASES.index((Z, A)) + ie
    sg, og = pm.nonelastic(Z, A, e_mev, n, seed)
    cg = pm.counters()
    so, oo = oracle_c1.nonelastic(Z, A, e_mev, n, seed + 5)
    # exact integers: charge and baryon number of every event (bit-exact bar)
    assert cg["n_zab_violations"] == 0
    # Reading R6.8: the step guard and the fixed capacities of the CUDA cascade (16 waiting / 16 outgoing nucleons) end
    # fewer than 1e-5 of the attempts, and the depth actually reached is the oracle's (7 in 1e6 events), far below them
    assert cg["n_inc_guard_trips"] + cg["n_inc_cap_trips"] <= max(1, 2e-5 * cg["n_inc_tries"]), cg
    assert 2 <= cg["inc_max_stack"] <= 10 and 2 <= cg["inc_max_out"] <= 10, cg
    zs = np.add.reduceat(sg["Z"].astype(np.int64), og[:-1]); as_ = np.add.reduceat(sg["A"].astype(np.int64), og[:-1])
    assert np.all(zs == Z + 1) and np.all(as_ == A + 1)
    assert og[0] == 0 and og[-1] == len(sg) and np.all(np.diff(og.astype(np.int64)) >= 2)
    assert np.all(sg[og[1:] - 1]["origin"] == 2)
    assert np.all(sg["ke"] >= 0) and np.allclose(np.linalg.norm(sg["dir"], axis=1), 1.0, atol=1e-4)
    # energy bookkeeping per event from the public records: nothing is created
    m = tables["nuclear_mass"]
    e_out = np.add.reduceat(sg["ke"].astype(np.float64) + m[sg["Z"], sg["A"]], og[:-1])
    left = e_mev + 938.27208816 + m[Z, A] - e_out
    assert np.all(left > -2e-2) and abs(left.sum() - cg["e_gamma"]) < 2e-2 * n
    # yields per species within 3 sigma (north_star), per origin
    yg, yo = parity.species_yields(sg, og), parity.species_yields(so, oo)
    err = np.sqrt(yg.var(axis=0) / n + yo.var(axis=0) / n)
    z = (yg.mean(axis=0) - yo.mean(axis=0)) / np.maximum(err, 1e-12)
    assert np.all(np.abs(z) < 3.0 + 0.5), (z, yg.mean(axis=0), yo.mean(axis=0))   # 48 comparisons: 3 sigma + look-elsewhere
    assert np.all(np.abs(yg.mean(axis=0) - yo.mean(axis=0)) <= 0.01 * yo.mean(axis=0) + 3.5 * err)
    # INC attempts per event (L75 restart rule)
    # (the number of tries is geometric: variance m(m-1) per event; 5 sigma of the difference of the two means)
    mt = oracle_c1.counters()["n_inc_tries"] / n
    assert abs(cg["n_inc_tries"] / n - mt) < 5 * np.sqrt(2 * mt * max(mt - 1, 0.01) / n)
    # spectra (5 MeV bins) and angles (20 bins), per species and origin
    for (zz, aa) in [(0, 1), (1, 1), (2, 4)]:
        for origin in (0, 1):
            a = sg[(sg["Z"] == zz) & (sg["A"] == aa) & (sg["origin"] == origin)]
            b = so[(so["Z"] == zz) & (so["A"] == aa) & (so["origin"] == origin)]
            if len(b) < 2000:
                continue
            c2, nb = parity.chi2_hist(a["ke"], b["ke"], np.arange(0.0, e_mev + 10.0, 5.0))
            assert c2 < 1 + 5 * np.sqrt(2.0 / max(nb, 1)), ("ke", zz, aa, origin, c2, nb)
            c2, nb = parity.chi2_hist(a["dir"][:, 2], b["dir"][:, 2], np.linspace(-1, 1, 21))
            assert c2 < 1 + 5 * np.sqrt(2.0 / max(nb, 1)), ("cos", zz, aa, origin, c2, nb)
    # residual (Z, A) map
    ra, rb = sg[og[1:] - 1], so[oo[1:] - 1]
    ka, kb = ra["Z"].astype(np.int64) * 64 + ra["A"], rb["Z"].astype(np.int64) * 64 + rb["A"]
    c2, nb = parity.chi2_hist(ka, kb, np.arange(-0.5, 64 * 24))
    assert c2 < 1 + 5 * np.sqrt(2.0 / max(nb, 1)), ("residual map", c2, nb)


def test_nonelastic_edge_cases(pm):
    from paper_1409_8336_b200 import PmcError
    sec, off = pm.nonelastic(8, 16, 200.0, 1, 3)                          # a single event
    assert len(off) == 2 and off[1] == len(sec) >= 2
    with pytest.raises(PmcError) as e:                                    # capacity too small: error, nothing silent
        pm.nonelastic(8, 16, 200.0, 1000, 3, capacity=100)
    assert e.value.code == -3
    with pytest.raises(PmcError) as e:                                    # hydrogen has no cascade
        pm.nonelastic(1, 1, 200.0, 10, 3)
    assert e.value.code == -5
    sec, off = pm.nonelastic(8, 16, 200.0, 0, 3)                          # no events at all
    assert len(sec) == 0 and len(off) == 1 and off[0] == 0
    # reproducible: same seed -> identical records; event i depends only on (seed, i)
    a, oa = pm.nonelastic(20, 40, 100.0, 5000, 9)
    b, ob_ = pm.nonelastic(20, 40, 100.0, 2500, 9)
    assert np.array_equal(oa[:2501], ob_) and a[:ob_[-1]].tobytes() == b.tobytes()


# ------------------------------------------------------------------ full path: dose parity (configs C1, C3, C4)
def _ledger_closes(c, rel=2e-4):
    sinks = c["e_deposit"] + c["e_escape"] + c["e_neutron"] + c["e_gamma"] + c["e_q"] + c["e_air"]
    return abs(sinks / c["e_source"] - 1) < rel


# The z statistic (D_gpu - D_oracle)/sqrt(sigma_g^2 + sigma_o^2) with both sigmas estimated from B batches is t-like: with
# B = 10 only 99.25 % of the voxels fall within 3 under PERFECT parity (99.66 % with 50 batches), and the
# pass fraction over nv voxels scatters binomially around that.  north_star's ">= 99 %" is therefore asserted literally
# with B = 40 batches on both sides (SURVEY's own remedy: "keep B a run-time option"), and where a configuration fixes
# B = 10 the bound is the expectation minus three binomial sigmas (voxels that share histories count as one in eight).
def low_stat_bound(nv, expect=0.9925):
    return expect - 3.0 * np.sqrt(expect * (1 - expect) / max(nv / 8.0, 1.0))


def _cascade_capacities_hold(cg, tag=""):
    """Reading R6.8 inside pmc_simulate (all the targets of the phantom, every energy the beam reaches): the fixed
    capacities of the CUDA cascade (16 waiting / 16 outgoing nucleons; the oracle allows 200 / any number) and its step
    guard end at most 1e-5 of the attempts, so the redraw they cause cannot bias the high-multiplicity events."""
    if cg["n_inc_tries"] == 0:
        return True
    print(f"cascade{tag}: {cg['n_inc_tries']} attempts, capacity trips {cg['n_inc_cap_trips']}, guard trips "
          f"{cg['n_inc_guard_trips']}, deepest stack {cg['inc_max_stack']}, most outgoing {cg['inc_max_out']}")
    return cg["n_inc_cap_trips"] + cg["n_inc_guard_trips"] <= max(1, 1e-5 * cg["n_inc_tries"])


def _dose_parity(pm, o, w_hu, vox, mats, spots, n, seed, axis=0, check_range=True, min_pass=0.99, batches=40, seed_o=None):
    """north_star's dose tolerances between pmc_simulate and the oracle on the same inputs (B batches on both sides).
    The oracle runs another seed (seed + 1000 unless given): with the same seed both sides draw the spot and the lateral
    position of every primary from the same Philox words, which correlates the two dose maps (rms z 0.82-0.92 was seen)
    and makes the comparison look better than it is.  rms z is held to a window around 1 for that reason."""
    if seed_o is None:
        seed_o = seed + 1000
    pm.set_option("n_batches", float(batches)); o.set_option("n_batches", float(batches))
    try:
        dg, sg = pm.simulate(spots, n, seed)
        cg = pm.counters()
        dg, sg = dg.cpu().numpy().astype(np.float64), sg.cpu().numpy().astype(np.float64)
        do, so = o.simulate(spots, n, seed_o)
        co = o.counters()
    finally:
        pm.set_option("n_batches", 10.0); o.set_option("n_batches", 10.0)
    assert np.all(np.isfinite(dg)) and np.all(dg >= 0) and np.all(sg >= 0)
    # integrated dose (= deposited energy per history) within 0.5 %
    rho = _density(w_hu, mats)
    vol = vox[0] * vox[1] * vox[2]
    eg, eo = (dg * rho).sum() * vol / parity.GY_PER_MEV_G, (do * rho).sum() * vol / parity.GY_PER_MEV_G
    # north_star's 0.5 %, plus three standard errors of the difference of two independent runs: with nuclear events on the
    # energy a history deposits has an rms of ~15 % of its mean (one in five loses tens of MeV to neutrons and photons),
    # i.e. 0.2 % on the difference at the 1e4 histories of C1 as configured, 0.02 % at 1e6
    assert abs(eg / eo - 1) < 5e-3 + 3 * 0.15 * np.sqrt(2.0 / n), (eg, eo)
    assert abs(eg - cg["e_deposit"] / n) < 2e-4 * eg                       # tally == ledger (fp32 atomics)
    assert _ledger_closes(cg), cg
    assert _cascade_capacities_hold(cg), cg
    # >= 99 % of voxels above 10 % of the maximum within 3 combined sigma
    frac, zmean, zrms, nv = parity.zscore_pass(dg, sg, do, so)
    if min_pass is None:
        min_pass = low_stat_bound(nv)
    else:            # the literal 99 % wherever the voxel count carries it (nv > ~5000); P(|t| < 3) = 99.6 % at B = 40
        min_pass = min(min_pass, low_stat_bound(nv, expect=0.996))
    print(f"z-pass {frac:.4f} (bound {min_pass:.4f}) mean z {zmean:+.3f} rms z {zrms:.3f} voxels {nv} B {batches} n {n}")
    assert nv > 20 and frac >= min_pass, (frac, zmean, zrms, nv)
    # independent runs: z has unit variance (t-like with 2(B - 1) degrees of freedom: 1.03 at B = 40, 1.12 at B = 10); the
    # voxels of a beam share histories (count one in eight), so rms z over nv voxels scatters by 2 / sqrt(nv)
    z_lo, z_hi = 0.95 - 6.0 / np.sqrt(nv), (1.2 if batches >= 30 else 1.3) + 6.0 / np.sqrt(nv)
    if seed_o == seed:
        z_lo = 0.0           # the same positions on both sides on purpose (deterministic case): no lower bound
    assert abs(zmean) < 0.25 and z_lo < zrms < z_hi, (zmean, zrms, z_lo, z_hi)
    # R80 and distal fall-off within 0.2 mm
    if check_range:
        d_cm = vox[2 - axis]
        r_g, f_g = parity.r80_and_falloff(parity.depth_dose(dg * rho, axis), d_cm)
        r_o, f_o = parity.r80_and_falloff(parity.depth_dose(do * rho, axis), d_cm)
        assert abs(r_g - r_o) < 0.02 and abs(f_g - f_o) < 0.02, (r_g, r_o, f_g, f_o)
    # event rates per history: statistically equal (Poisson)
    for k in ("n_elastic", "n_nonelastic", "n_secondary_protons"):
        a, b = cg[k], co[k]
        assert abs(a - b) < 5 * np.sqrt(a + b + 1) + 0.002 * b, (k, a, b)
    # steps per history: rms ~ 30 % of the mean (a non-elastic event ends the primary anywhere along its track)
    assert abs(cg["n_steps"] / co["n_steps"] - 1) < 5e-3 + 3 * 0.3 * np.sqrt(2.0 / n)
    return dg, sg, do, so, cg, co


def _density(hu, mats):
    rho = np.zeros(hu.shape)
    h = hu.astype(np.float64)
    for i, m in enumerate(mats):
        lo = -np.inf if i == 0 else m["hu_lo"]
        hi = np.inf if i == len(mats) - 1 else m["hu_hi"]
        sel = (h >= lo) & (h < hi)
        t = np.clip(h[sel], m["hu_lo"], m["hu_hi"])
        rho[sel] = m["rho_lo"] + (m["rho_hi"] - m["rho_lo"]) * (t - m["hu_lo"]) / (m["hu_hi"] - m["hu_lo"])
    return rho


def test_c1_water_phantom_as_configured(pm, tables):
    """C1 exactly as BASELINE.json configures it (1e4 histories, seed 1, 10 batches): bound of SURVEY 8(c).8 at B = 10; the
    same 1e4 histories with 40 batches: north_star's literal 99 %."""
    w = inputs.workload("c1")                                             # 1e4 histories, seed 1, full physics
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    _dose_parity(pm, o, w["hu"], w["vox"], w["materials"], w["spots"], w["n_histories"], w["seed"], min_pass=None, batches=10)
    _dose_parity(pm, o, w["hu"], w["vox"], w["materials"], w["spots"], w["n_histories"], w["seed"])


def _lateral_width(d, k):
    p = d[k - 5:k + 1].sum(axis=(0, 1)); x = np.arange(len(p))
    return np.sqrt((p * (x - (p * x).sum() / p.sum()) ** 2).sum() / p.sum())


def test_c1_water_phantom_high_statistics(pm, tables):
    """C1 at 3e6 histories (the paper's own pencil-beam statistics are 2.6e6), 30 batches, different seeds
    on the two sides: every north_star tolerance at once, plus the lateral width at the Bragg peak (MCS + nuclear halo)
    and the ledgers."""
    w = inputs.workload("c1")
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    dg, sg, do, so, cg, co = _dose_parity(pm, o, w["hu"], w["vox"], w["materials"], w["spots"], 3_000_000, 11, batches=30, seed_o=12)
    k = int(np.argmax(do.sum(axis=(1, 2))))
    assert abs(_lateral_width(dg, k) / _lateral_width(do, k) - 1) < 3e-3
    for key in ("e_neutron", "e_gamma", "e_q", "e_escape"):
        assert abs(cg[key] / co[key] - 1) < 0.01, (key, cg[key], co[key])


@pytest.mark.parametrize("switches", [dict(straggling=0, mcs=0, elastic=0, nonelastic=0),
                                      dict(elastic=0, nonelastic=0), dict(nonelastic=0), dict(elastic=0)])
def test_c1_physics_switches(pm, tables, switches):
    w = inputs.workload("c1")
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"], **switches)
    # With every fluctuation off all histories are the same CSDA track and only the spot position is random: the voxels
    # of a column then fluctuate together (a handful of independent z values, not 475), so that case is compared with the
    # SAME seed on both sides - the same positions, hence the same dose up to fp32 (rms z ~ 0.001) - a deterministic check.
    same = "mcs" in switches and "straggling" in switches
    _dose_parity(pm, o, w["hu"], w["vox"], w["materials"], w["spots"], 100_000, 21, seed_o=21 if same else None)


def test_pencil_on_a_voxel_edge(pm, tables):
    """A zero-width pencil aimed exactly at the common edge of four voxel columns (x = y = 5.0 cm on the 2 mm grid).  Which of
    the four voxels a start point on a face belongs to is decided by each side's own arithmetic (the oracle divides by
    0.2 in fp64, the sampler by float(0.2)); Reading R3.8 makes that immaterial: a proton that is deflected away from its
    voxel crosses the face in a zero-length boundary step.  So the dose must agree like anywhere else, and be symmetric
    about the edge on both sides."""
    w = inputs.workload("c1")
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    spot = inputs.plan_single_spot((5.0, 5.0, 0.0), 150.0, 0.0)
    dg, sg, do, so, cg, co = _dose_parity(pm, o, w["hu"], w["vox"], w["materials"], spot, 400_000, 61, seed_o=62)
    # Every step scores in the voxel it starts in, and a proton deflected towards a face it sits on crosses it at once and
    # is deflected afresh in the next voxel: for a pencil of zero width on an edge the four columns around it therefore get
    # slightly different doses (4 % more in the voxel that owns the start point, 1 % between the two mirror columns because
    # x faces are met before y faces, Reading R3.2) - artefacts of the class II scheme of a few micrometres, identical on
    # both sides because the tie rules are (start point: upper voxel, placed in fp64; faces: x before y before z).  What
    # parity asks: each of the four columns agrees within its statistical error, and so does the excess of the owner.
    # (the slabs of a column are crossed by the same protons, so their errors add linearly, not in quadrature)
    cg_, co_ = dg[:70].sum(axis=0), do[:70].sum(axis=0)
    eg_, eo_ = sg[:70].sum(axis=0), so[:70].sum(axis=0)
    for a in ((24, 24), (24, 25), (25, 24), (25, 25)):
        assert abs(cg_[a] - co_[a]) < 3.0 * np.hypot(eg_[a], eo_[a]), (a, cg_[a], co_[a], eg_[a], eo_[a])
    assert cg_[25, 25] / cg_[24, 24] > 1.02 and co_[25, 25] / co_[24, 24] > 1.02
    # first steps from the edge: after 30 steps the transverse distribution is symmetric and equal on both sides
    for k_ in ("elastic", "nonelastic"):
        pm.set_option(k_, 0.0); o.set_option(k_, 0.0)
    g = pm.first_steps(spot, 100_000, 5, 30).astype(np.float64); r = o.first_steps(spot, 100_000, 6, 30)
    for col in (0, 1):
        assert abs(g[:, col].mean() - 5.0) < 5 * g[:, col].std() / np.sqrt(1e5) and abs(r[:, col].mean() - 5.0) < 5 * r[:, col].std() / np.sqrt(1e5)
        assert abs(g[:, col].std() / r[:, col].std() - 1) < 0.02


@pytest.mark.parametrize("name", ["c3_70", "c3_150", "c3_230"])
def test_c3_slab_phantom(pm, tables, name):
    w = inputs.workload(name)                                             # full 200x200x300 grid, 24-bin table
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    # as configured: 1e6 histories per energy (BASELINE.json C3), other seed on the oracle side
    # 230 MeV leaves the 30 cm slab: no Bragg peak inside, so no R80
    dg, sg, do, so, cg, co = _dose_parity(pm, o, w["hu"], w["vox"], w["materials"], w["spots"], w["n_histories"], w["seed"],
                                          check_range=(name != "c3_230"), seed_o=w["seed"] + 100)
    if name == "c3_230":
        assert abs(cg["e_escape"] / co["e_escape"] - 1) < 5e-3
    # energy deposited per material class (water / bone / lung / Ti)
    rho = _density(w["hu"], w["materials"])
    for lo, hi in [(-5, 6), (1200, 1201), (-700, -699), (3071, 3072)]:
        m = (w["hu"] >= lo) & (w["hu"] < hi)
        a, b = (dg * rho)[m].sum(), (do * rho)[m].sum()
        if b > 0:
            assert abs(a / b - 1) < 1e-2, (lo, a, b)


def test_c4_head_and_neck_at_full_size_on_both_sides(pm, tables):
    """north_star's target: C4 with 1e7 histories on the CUDA path AND on the oracle (different seeds), with the stated
    tolerances: integrated dose 0.5 %, >= 99 % of the voxels above 10 % of the maximum within 3 combined sigma (asserted
    with 40 batches on both sides; the CUDA path is also run with the configured 10 batches and that pass rate reported
    and bounded).  Dose to air is left out of the voxel comparison (Reading R8.1 in DESIGN.md: with rho = 0.0012 g/cm3 a
    voxel of air turns a single stopping proton into a dose a thousand times that of tissue, so the 'maximum dose' of the
    grid would be set by one such voxel); the pass rate over ALL voxels is computed and bounded as well."""
    w = inputs.workload("c4")
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    n = w["n_histories"]
    rho = _density(w["hu"], w["materials"]); vol = np.prod(w["vox"]); tissue = w["hu"] >= -950
    pm.set_option("n_batches", 40.0); o.set_option("n_batches", 40.0)
    try:
        dg, sg = pm.simulate(w["spots"], n, w["seed"]); cg = pm.counters()
        dg, sg = dg.cpu().numpy().astype(np.float64), sg.cpu().numpy().astype(np.float64)
        do, so = o.simulate(w["spots"], n, w["seed"] + 1); co = o.counters()
    finally:
        pm.set_option("n_batches", 10.0); o.set_option("n_batches", 10.0)
    d10, s10 = pm.simulate(w["spots"], n, w["seed"])                    # the configured 10 batches, same histories
    d10, s10 = d10.cpu().numpy().astype(np.float64), s10.cpu().numpy().astype(np.float64)
    assert _ledger_closes(cg) and cg["n_zab_violations"] == 0 and co["n_zab_violations"] == 0
    assert _cascade_capacities_hold(cg, " C4") and cg["inc_max_stack"] < 16 and cg["inc_max_out"] < 16, cg
    assert np.allclose(d10[tissue], dg[tissue], rtol=3e-4, atol=1e-16)  # the batch split does not change the dose
    eg, eo = (dg * rho).sum() * vol / parity.GY_PER_MEV_G, (do * rho).sum() * vol / parity.GY_PER_MEV_G
    assert abs(eg / eo - 1) < 5e-3 and abs(eg / eo - 1) < 1e-3, (eg, eo)             # integrated dose (0.5 % asked; 0.1 % seen)
    assert abs(eg - cg["e_deposit"] / n) < 3e-4 * eg
    for k in ("n_steps", "n_elastic", "n_nonelastic", "n_secondary_protons", "n_missed"):
        a, b = cg[k], co[k]
        assert abs(a - b) <= 5 * np.sqrt(a + b + 1) + 2e-3 * b, (k, a, b)
    for k in ("e_neutron", "e_gamma", "e_q", "e_escape", "e_air"):
        assert abs(cg[k] / co[k] - 1) < 0.01, (k, cg[k], co[k])
    frac, zmean, zrms, nv = parity.zscore_pass(dg, sg, do, so, region=tissue)
    f_all, zm_all, zr_all, nv_all = parity.zscore_pass(dg, sg, do, so)
    f10, zm10, zr10, nv10 = parity.zscore_pass(d10, s10, do, so, region=tissue)
    print(f"C4 1e7 vs 1e7: tissue z-pass {frac:.4f} (mean {zmean:+.3f} rms {zrms:.3f}, {nv} voxels); all voxels {f_all:.4f} "
          f"({nv_all}); CUDA path at B = 10: {f10:.4f}; integrated dose ratio - 1 = {eg / eo - 1:+.2e}")
    assert nv > 30_000 and frac >= 0.99 and abs(zmean) < 0.1 and zrms < 1.15, (frac, zmean, zrms, nv)
    assert f10 >= 0.99 - 0.003 and f_all >= 0.985, (f10, f_all)
    # the three 1-D projections of deposited energy, slab by slab
    # every slab above 5 % of the largest one.  The statistical error of a slab sum (its voxels share histories, so the voxel
    # sigmas cannot simply be added) is measured: the scatter of twelve more 1e7-history runs of the CUDA path with other seeds (variance smoothed over
    # nine neighbouring slabs; thirteen runs alone leave the per-slab sigma uncertain by 20 %).
    prof_g = [[parity.depth_dose(dg * rho, ax) for ax in range(3)]]
    for k in range(12):
        dk, _ = pm.simulate(w["spots"], n, 7000 + k)
        dk = dk.cpu().numpy().astype(np.float64) * rho
        prof_g.append([parity.depth_dose(dk, ax) for ax in range(3)])
    for ax in range(3):
        runs = np.array([p_[ax] for p_ in prof_g]); po = parity.depth_dose(do * rho, ax)
        mean = runs.mean(axis=0)
        rel_var = np.convolve(runs.var(axis=0, ddof=1) / np.maximum(mean, 1e-300) ** 2, np.ones(9) / 9, mode="same")
        sd = np.sqrt(rel_var) * mean
        m = po > 0.05 * po.max()
        zz = (mean[m] - po[m]) / (sd[m] * np.sqrt(1 + 1 / 13.0))
        print(f"PROJ axis {ax}: max |z| {np.abs(zz).max():.2f} mean z {zz.mean():+.2f} rms z {zz.std():.2f} max rel diff {np.max(np.abs(mean[m] / po[m] - 1)):.2e}")
        assert np.all(np.abs(mean[m] - po[m]) < 4.5 * sd[m] * np.sqrt(1 + 1 / 13.0) + 1e-3 * po[m]), (ax, np.abs(zz).max())
        assert np.all(np.abs(mean[m] / po[m] - 1) < 2e-2)
    # sigma: same number of histories, same sigma (median relative error in the high-dose region)
    hi = tissue & (do > 0.5 * do[tissue].max())
    assert abs(np.median(sg[hi] / dg[hi]) / np.median(so[hi] / do[hi]) - 1) < 0.05


@pytest.mark.parametrize("field", [0, 1, 2])
def test_c4_range_of_each_field_along_its_own_axis(pm, tables, field):
    """R80 and distal fall-off (R20 - R80) within 0.2 mm on the integrated depth dose of each of the three C4 fields along
    its own axis (+x, -x, -y), each field's spots simulated separately with 2e6 histories on both sides.  The distal edge of
    a multi-layer field is searched from the far end of the profile (its plateau has no usable maximum)."""
    w = inputs.workload("c4")
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    dirs = np.array([(1.0, 0.0, 0.0), (-1.0, 0.0, 0.0), (0.0, -1.0, 0.0)])
    sel = np.all(np.abs(w["spots"][:, 3:6] - dirs[field]) < 1e-9, axis=1)
    spots = np.ascontiguousarray(w["spots"][sel])
    assert 300 < len(spots) < 1500
    n = 2_000_000
    dg, _ = pm.simulate(spots, n, 400 + field); dg = dg.cpu().numpy().astype(np.float64)
    do, _ = o.simulate(spots, n, 500 + field)
    rho = _density(w["hu"], w["materials"])
    axis = 2 if field < 2 else 1; d_cm = w["vox"][0] if field < 2 else w["vox"][1]
    pg, po = parity.depth_dose(dg * rho, axis), parity.depth_dose(do * rho, axis)
    if dirs[field][0 if field < 2 else 1] < 0:
        pg, po = pg[::-1], po[::-1]
    assert abs(pg.sum() / po.sum() - 1) < 5e-3
    r80g, r80o = parity.distal_depth_from_end(pg, d_cm, 0.8), parity.distal_depth_from_end(po, d_cm, 0.8)
    r20g, r20o = parity.distal_depth_from_end(pg, d_cm, 0.2), parity.distal_depth_from_end(po, d_cm, 0.2)
    print(f"C4 field {field}: R80 {r80g:.4f} vs {r80o:.4f} cm, fall-off {10 * (r20g - r80g):.3f} vs {10 * (r20o - r80o):.3f} mm")
    assert np.isfinite([r80g, r80o, r20g, r20o]).all()
    assert abs(r80g - r80o) < 0.02 and abs((r20g - r80g) - (r20o - r80o)) < 0.02


def test_c4_two_seeds_eq5_and_gamma(pm, tables):
    """PAPER.md:L172 Eq.5: two runs that differ only in the seed scatter by sqrt(2) x the reported statistical error;
    and their 3-D gamma index (2 %/2 mm, L166) passes everywhere.  Pins the batch sigma of the CUDA path at full size."""
    w = inputs.workload("c4")
    _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    n = w["n_histories"]
    d1, s1 = pm.simulate(w["spots"], n, 101); d1, s1 = d1.clone(), s1.clone()
    d2, s2 = pm.simulate(w["spots"], n, 202)
    tissue = torch.as_tensor(w["hu"] >= -950, device=d1.device)
    hi = tissue & (d1 > 0.5 * d1[tissue].max())
    assert int(hi.sum()) > 1000
    delta = ((d1[hi] - d2[hi]) / d1[hi]).double()
    sig = (0.5 * (s1[hi] / d1[hi] + s2[hi] / d2[hi])).double()
    ratio = float(delta.pow(2).mean().sqrt() / (np.sqrt(2.0) * sig.pow(2).mean().sqrt()))
    assert abs(ratio - 1) < 0.1, ratio                                     # 10-batch sigma estimator, RMS over > 1e3 voxels
    a, b = d1 * tissue, d2 * tissue                                        # dose to tissue (air voxels spike, see above)
    g, rate = pm.gamma_index(a, b, w["vox"], 0.02, 0.2, 0.1)
    assert rate > 0.995 and float(g.max()) < 3.0, rate


def test_c5_pelvis_full_size_against_oracle_subsample(pm, tables):
    """C5 (512x512x200 pelvis with Ti implants, 11033 spots, 100-230 MeV) at BASELINE's full 1e8 histories on the GPU
    (6 sub-groups of 2^24 histories); the oracle runs a 1e7-history subsample (ten times what SURVEY 8(d) assigns to this
    throughput configuration, so that its own noise in low-count voxels no longer skews the z scores).  40 batches on both sides for the voxel comparison (see low_stat_bound above)."""
    w = inputs.workload("c5")
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    n_g, n_o = w["n_histories"], 10_000_000
    pm.set_option("n_batches", 40.0); o.set_option("n_batches", 40.0)
    try:
        dg, sg = pm.simulate(w["spots"], n_g, w["seed"])
        cg = pm.counters()
        dg, sg = dg.cpu().numpy().astype(np.float64), sg.cpu().numpy().astype(np.float64)
        do, so = o.simulate(w["spots"], n_o, w["seed"] + 1)
        co = o.counters()
    finally:
        pm.set_option("n_batches", 10.0); o.set_option("n_batches", 10.0)
    assert _ledger_closes(cg) and cg["n_zab_violations"] == 0 and np.all(np.isfinite(dg)) and np.all(sg >= 0)
    assert _cascade_capacities_hold(cg, " C5") and cg["inc_max_stack"] < 16 and cg["inc_max_out"] < 16, cg
    rho = _density(w["hu"], w["materials"])
    vol = np.prod(w["vox"])
    eg, eo = (dg * rho).sum() * vol / parity.GY_PER_MEV_G, (do * rho).sum() * vol / parity.GY_PER_MEV_G
    assert abs(eg / eo - 1) < 5e-3                                         # integrated dose 0.5 %
    assert abs(eg - cg["e_deposit"] / n_g) < 3e-4 * eg
    for k in ("n_steps", "n_elastic", "n_nonelastic", "n_secondary_protons", "n_missed"):
        a, b = cg[k] / n_g, co[k] / n_o
        assert abs(a - b) <= 5 * np.sqrt(b / n_o + a / n_g) + 5e-3 * b, (k, a, b)
    # energy deposited in the titanium implants (own stopping-power table, HU clamp 3071 -> 4.5 g/cm3, L49)
    ti = w["hu"] >= 3060
    a, b = (dg * rho)[ti].sum(), (do * rho)[ti].sum()
    assert b > 0 and abs(a / b - 1) < 0.03, (a, b)
    # voxel z-scores in tissue and bone (not air, Reading R8.1)
    frac, zmean, zrms, nv = parity.zscore_pass(dg, sg, do, so, region=w["hu"] >= -950)
    print(f"C5 1e8 vs oracle 1e7: z-pass {frac:.4f} mean z {zmean:+.3f} rms z {zrms:.3f} voxels {nv}")
    # mean z: +0.120 against a 1e6-history oracle run, +0.067 against 1e7 - it falls as the ORACLE's statistics improve
    # (skewed low-count voxels of the sparser run), where a bias of the CUDA path would grow in units of the shrinking sigma;
    # C4 with 1e7 histories on both sides has +0.008
    assert nv > 100_000 and frac >= 0.99 and abs(zmean) < 0.1 and 0.95 < zrms < 1.2, (frac, zmean, zrms, nv)
    for ax in range(3):
        pg, po = parity.depth_dose(dg * rho, ax), parity.depth_dose(do * rho, ax)
        m = po > 0.05 * po.max()
        tol = 0.01 + 0.012 * np.sqrt(po.max() / po[m])
        assert np.all(np.abs(pg[m] / po[m] - 1) < tol), (ax, np.max(np.abs(pg[m] / po[m] - 1) / tol))


# ------------------------------------------------------------------ LET_d scoring
def test_letd_deterministic_column_matches_oracle(pm, tables):
    # fluctuations off: every history is the same CSDA track, LET_d per slab compared element by element
    hu, vox = np.zeros((100, 1, 1), dtype=np.int16), (50.0, 50.0, 0.2)
    o = _setup(pm, tables, inputs.make_materials_c1(), hu, vox, straggling=0, mcs=0, elastic=0, nonelastic=0)
    spot = inputs.plan_single_spot((25.0, 25.0, 0.0), 150.0, 0.0)
    pm.set_option("score_letd", 1.0); o.set_option("score_letd", 1.0)
    try:
        pm.simulate(spot, 64, 3); o.simulate(spot, 64, 3)
        lg, lo = pm.letd().cpu().numpy().astype(np.float64)[:, 0, 0], o.letd()[:, 0, 0]
    finally:
        pm.set_option("score_letd", 0.0)
    k_end = int(np.max(np.nonzero(lo)[0]))
    assert np.all(lg[k_end + 1:] == 0) and np.all(lo[k_end + 1:] == 0)
    assert np.max(np.abs(lg[:k_end - 1] / lo[:k_end - 1] - 1)) < 2e-4      # fp32 range-table differences per slab
    assert abs(lg[k_end] / lo[k_end] - 1) < 0.05                          # the stopping slab: e0 / residual range


def test_letd_full_physics_matches_oracle(pm, tables):
    from paper_1409_8336_b200 import PmcError
    w = inputs.workload("c1")
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    n = 200_000
    with pytest.raises(PmcError) as e:                                    # nothing scored yet
        pm.simulate(w["spots"], 100, 1); pm.letd()
    assert e.value.code == -2
    d0, _ = pm.simulate(w["spots"], n, 31)
    pm.set_option("score_letd", 1.0); o.set_option("score_letd", 1.0)
    try:
        dg, _ = pm.simulate(w["spots"], n, 31); lg = pm.letd().cpu().numpy().astype(np.float64)
        do, _ = o.simulate(w["spots"], n, 32); lo = o.letd()
        do2, _ = o.simulate(w["spots"], n, 33); lo2 = o.letd()             # second oracle run: the noise yardstick
    finally:
        pm.set_option("score_letd", 0.0)
    assert torch.allclose(dg, d0, rtol=2e-4, atol=1e-16)                  # scoring LET_d does not change the dose
    dg = dg.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(lg)) and np.all(lg >= 0) and np.all((lg > 0) <= (dg > 0))
    # dose-weighted LET_d per slab, up to the distal 10 % of the depth dose
    def prof(l, d):
        return (l * d).sum(axis=(1, 2)) / np.maximum(d.sum(axis=(1, 2)), 1e-300)
    pg, po, po2 = prof(lg, dg), prof(lo, do), prof(lo2, do2)
    dd = do.sum(axis=(1, 2)); m = dd > 0.1 * dd.max()
    # noise yardstick: the oracle-vs-oracle difference, as the largest over a window of +-3 slabs (a few soft secondary
    # protons of very high LET dominate the entrance slabs, so the scatter of a single slab is itself very noisy)
    noise = np.abs(po2[m] / po[m] - 1)
    noise = np.array([noise[max(0, i - 3):i + 4].max() for i in range(len(noise))])
    assert np.all(np.abs(pg[m] / po[m] - 1) < 0.01 + 4 * np.maximum(noise, np.median(noise))), (pg[m] / po[m])[:80]
    assert abs(np.mean(pg[m] / po[m]) - 1) < 3e-3                         # no systematic offset along the depth
    # voxel by voxel in the high-dose region: GPU-vs-oracle scatter is the oracle-vs-oracle scatter
    hi = do > 0.1 * do.max()
    rg, ro = lg[hi] / lo[hi] - 1, lo2[hi] / lo[hi] - 1
    assert abs(np.median(rg)) < 3e-3 and rg.std() < 1.25 * ro.std() + 1e-3, (np.median(rg), rg.std(), ro.std())


# ------------------------------------------------------------------ per-spot dose influence
def test_dose_influence_matches_oracle(pm, tables):
    from paper_1409_8336_b200 import PmcError
    w = inputs.workload("c1")
    hu, vox = w["hu"], w["vox"]
    o = _setup(pm, tables, w["materials"], hu, vox)
    nz, ny, nx = hu.shape
    a = inputs.plan_single_spot((3.0, 5.0, 0.0), 100.0, 0.3); b = inputs.plan_single_spot((7.0, 5.0, 0.0), 150.0, 0.3)
    c = inputs.plan_single_spot((5.0, 5.0, 0.0), 120.0, 0.3); d = inputs.plan_single_spot((5.0, 5.0, 0.0), 70.0, 0.5)
    spots = np.concatenate([a, b, c, d]); spots[:, 12] = [1.0, 2.0, 0.0, 1.0]
    # ROI: a 7 x 7 column around each of the three beam axes, every second slab, shuffled
    cols = [(x, y) for cx in (15, 25, 35) for x in range(cx - 3, cx + 4) for y in range(22, 29)]
    roi = np.array([(z * ny + y) * nx + x for z in range(0, nz, 2) for (x, y) in cols], dtype=np.int32)
    roi = np.random.default_rng(3).permutation(roi)
    n = 200_000                                                            # divisible by the 10 batches
    D = pm.set_dose_influence(roi, len(spots)); o.set_dose_influence(roi)
    try:
        dose, _ = pm.simulate(spots, n, 51)
        Dg = D.cpu().numpy().astype(np.float64)
        dose_o, _ = o.simulate(spots, n, 52)
        Do = o.dose_influence(len(spots))
        with pytest.raises(PmcError) as e:                                # more spots than the matrix has rows
            pm.simulate(np.concatenate([spots, spots]), 100, 1)
        assert e.value.code == -3
    finally:
        pm.set_dose_influence(np.zeros(0, dtype=np.int32), 0); o.set_dose_influence(np.zeros(0, dtype=np.int32))
    dg = dose.cpu().numpy().astype(np.float64).ravel()[roi]
    # exact bookkeeping on the GPU: the rows add up to the dose (fp32 atomics, two different summation orders)
    assert np.all(Dg >= 0) and np.all(Dg[2] == 0)
    assert np.allclose(Dg.sum(axis=0), dg, rtol=3e-4, atol=1e-6 * dg.max())
    # against the oracle, spot by spot: integral over the ROI, and the depth profile on the spot's own axis
    zz, xx = roi // (nx * ny), roi % nx
    for i, cx in ((0, 15), (1, 35), (3, 25)):
        assert abs(Dg[i].sum() / Do[i].sum() - 1) < 0.01, (i, Dg[i].sum(), Do[i].sum())
        own = np.abs(xx - cx) <= 3
        pg = np.bincount(zz[own], weights=Dg[i][own], minlength=nz)[::2]; po = np.bincount(zz[own], weights=Do[i][own], minlength=nz)[::2]
        m = po > 0.1 * po.max()
        assert np.max(np.abs(pg[m] / po[m] - 1)) < 0.04, (i, np.max(np.abs(pg[m] / po[m] - 1)))
        assert abs(int(np.argmax(pg)) - int(np.argmax(po))) <= 1           # each spot's Bragg peak where its energy puts it
        other = ~own & (np.abs(xx - 25) > 3 if i != 3 else np.abs(xx - 25) > 3)
        assert Dg[i][other].sum() < 0.02 * Dg[i].sum()                    # (almost) nothing on the other beams' axes
    # the dose itself is unchanged by the extra scoring
    d0, _ = pm.simulate(spots, n, 51)
    assert torch.allclose(d0, dose, rtol=2e-4, atol=1e-16)


# ------------------------------------------------------------------ full Moliere MCS option
def test_moliere_option_matches_oracle(pm, tables):
    from scipy import stats
    w = inputs.workload("c1")
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"], elastic=0, nonelastic=0, straggling=0)
    pm.set_option("mcs_model", 1.0); o.set_option("mcs_model", 1.0)
    try:
        # one 2 mm step at 150 MeV and at 70 MeV: the whole space-angle distribution, core and single-scattering tail
        for e_mev in (150.0, 70.0):
            spot = inputs.plan_single_spot((5.1, 5.1, 0.0), e_mev, 0.0)
            n = 400_000
            g = pm.first_steps(spot, n, 5, 1).astype(np.float64); r = o.first_steps(spot, n, 6, 1)
            tg, to = np.hypot(g[:, 3], g[:, 4]), np.hypot(r[:, 3], r[:, 4])
            assert stats.ks_2samp(tg, to).pvalue > 1e-3
            t0 = np.median(to)
            for mult in (3.0, 6.0, 12.0):                                  # tail counts: Poisson
                a, b = np.sum(tg > mult * t0), np.sum(to > mult * t0)
                assert abs(a - b) < 5 * np.sqrt(a + b + 1), (e_mev, mult, a, b)
            assert np.sum(to > 6.0 * t0) > 100                             # the tail is there (a Gaussian has e^-25)
        # 40 steps at 230 MeV: lateral spread and angle-displacement covariance of the multi-step walk
        spot = inputs.plan_single_spot((5.1, 5.1, 0.0), 230.0, 0.0)
        g = pm.first_steps(spot, 200_000, 5, 40).astype(np.float64); r = o.first_steps(spot, 200_000, 6, 40)
        for col in (0, 3):
            assert abs(np.percentile(np.abs(g[:, col] - (5.1 if col == 0 else 0)), 68.27) /
                       np.percentile(np.abs(r[:, col] - (5.1 if col == 0 else 0)), 68.27) - 1) < 0.02
        # full physics on C1 with the Moliere option on both sides
        for k in ("elastic", "nonelastic", "straggling"):
            pm.set_option(k, 1.0); o.set_option(k, 1.0)
        _dose_parity(pm, o, w["hu"], w["vox"], w["materials"], w["spots"], 100_000, 23)
        # without the tables the option is refused
        from paper_1409_8336_b200 import PmcError
    finally:
        pm.set_option("mcs_model", 0.0)
    with pytest.raises(PmcError):
        pm.set_option("mcs_model", 2.0)


# ------------------------------------------------------------------ edge and degenerate cases
def test_simulate_edge_cases(pm, tables):
    from paper_1409_8336_b200 import PmcError
    w = inputs.workload("c1")
    o = _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    # every history misses the grid: zero dose, energy all in the escape ledger
    away = inputs.plan_single_spot((50.0, 50.0, -5.0), 150.0, 0.1)
    d, s = pm.simulate(away, 1000, 1)
    c = pm.counters()
    assert float(d.abs().sum()) == 0.0 and float(s.abs().sum()) == 0.0
    assert c["n_missed"] == 1000 and c["n_steps"] == 0 and abs(c["e_escape"] - 150.0 * 1000) < 1e-6
    do, _ = o.simulate(away, 1000, 1)
    assert do.sum() == 0.0 and o.counters()["n_missed"] == 1000
    # fewer histories than batches (every group needs its N/10 histories): refused on both sides
    for n in (1, 7):
        with pytest.raises(PmcError) as e:
            pm.simulate(w["spots"], n, 3)
        assert e.value.code == -1
        with pytest.raises(RuntimeError):
            o.simulate(w["spots"], n, 3)
    # one history per batch: the dose grid integrates to the deposited energy per history
    d, s = pm.simulate(w["spots"], 10, 3)
    c = pm.counters()
    assert _ledger_closes(c) and abs(c["e_source"] - 150.0 * 10) < 1e-6
    e_grid = float(d.double().sum()) * 1.0 * 0.2 ** 3 / parity.GY_PER_MEV_G          # water, rho = 1
    assert abs(e_grid - c["e_deposit"] / 10) < 2e-4 * e_grid
    # air gap: source 20 cm upstream of the grid
    up = inputs.plan_single_spot((5.0, 5.0, -20.0), 150.0, 0.3)
    d, s = pm.simulate(up, 50_000, 5)
    cg = pm.counters()
    o.simulate(up, 50_000, 6)
    co = o.counters()
    assert cg["e_air"] > 0 and abs(cg["e_air"] / co["e_air"] - 1) < 0.02 and _ledger_closes(cg)
    # oblique beam entering through a side face
    ob_ = inputs.plan_single_spot((-3.0, 5.0, 6.0), 100.0, 0.3, direction=(0.8, 0.0, 0.6))
    _dose_parity(pm, o, w["hu"], w["vox"], w["materials"], ob_, 60_000, 8, check_range=False)
    # the smallest grid there is: one voxel, everything the protons lose before they leave is in it
    one = np.zeros((1, 1, 1), dtype=np.int16)
    pm.load_ct(torch.as_tensor(one, device="cuda"), (0.5, 0.5, 0.5)); o.load_ct(one, (0.5, 0.5, 0.5))
    mid = inputs.plan_single_spot((0.25, 0.25, 0.0), 150.0, 0.0)
    d1, _ = pm.simulate(mid, 20_000, 9); c1 = pm.counters()
    do1, _ = o.simulate(mid, 20_000, 10); co1 = o.counters()
    assert d1.shape == (1, 1, 1) and _ledger_closes(c1)
    assert abs(c1["e_deposit"] / co1["e_deposit"] - 1) < 0.02 and abs(c1["e_escape"] / co1["e_escape"] - 1) < 1e-3
    assert abs(float(d1[0, 0, 0]) / do1[0, 0, 0] - 1) < 0.02
    pm.load_ct(torch.as_tensor(w["hu"], device="cuda"), w["vox"]); o.load_ct(w["hu"], w["vox"])
    # zero-weight and bad inputs
    bad = w["spots"].copy(); bad[0, 12] = 0.0
    with pytest.raises(PmcError):
        pm.simulate(bad, 10, 1)
    bad = w["spots"].copy(); bad[0, 3:6] = 0.0
    with pytest.raises(PmcError):
        pm.simulate(bad, 10, 1)


def test_ragged_grid_and_clamped_hu(pm, tables):
    """Odd, anisotropic grid (37 x 23 x 41 voxels of 1.3 x 2.1 x 1.7 mm) with HU outside the table on both sides:
    below the first bin (-2000 -> air) and above the last (5000 -> the Ti bin, PAPER.md:L49 '>3060 = metal implant'),
    a bone slab and a lung slab; oblique beam.  Same clamping, indexing and face logic on both sides."""
    mats = inputs.make_materials_24()
    nz, ny, nx = 41, 23, 37
    hu = np.zeros((nz, ny, nx), dtype=np.int16)
    hu[:, :, :3] = -2000; hu[10:14] = 1200; hu[14:20] = -700; hu[24:27, 8:14, 14:22] = 5000
    vox = (0.13, 0.21, 0.17)
    o = _setup(pm, tables, mats, hu, vox)
    spot = inputs.plan_single_spot((2.4, 2.3, -1.0), 90.0, 0.25, direction=(0.05, 0.02, 1.0), sigma_e=0.8, div=0.004)
    dg, sg, do, so, cg, co = _dose_parity(pm, o, hu, vox, mats, spot, 120_000, 17, check_range=False)
    rho = _density(hu, mats)
    for sel in (hu == 5000, hu == 1200, hu == -700):
        a, b = (dg * rho)[sel].sum(), (do * rho)[sel].sum()
        assert b > 0 and abs(a / b - 1) < 1.5e-2, (a, b)
    assert cg["e_air"] > 0 and abs(cg["e_air"] / co["e_air"] - 1) < 0.02


def test_density_varies_inside_the_first_and_last_hu_bin(pm, tables):
    """Two water-like HU bins whose density is linear in HU (rho(HU) inside a bin), with HU values spread over
    both and beyond both ends of the table: the step kernel's per-HU density table holds one entry for each of the two end
    bins and must fall back to the bin's own line there."""
    water = inputs.make_materials_c1()[1]
    lo = dict(water, hu_lo=-600, hu_hi=0, rho_lo=0.4, rho_hi=1.0)
    hi = dict(water, hu_lo=0, hu_hi=1000, rho_lo=1.0, rho_hi=1.8)
    mats = [lo, hi]
    nz, ny, nx = 80, 21, 21
    hu = np.zeros((nz, ny, nx), dtype=np.int16)
    for k in range(nz):
        hu[k] = [-900, -500, -250, -1, 0, 300, 700, 999, 1500, -100][k % 10]      # -900 and 1500 are clamped to the end bins
    vox = (0.2, 0.2, 0.2)
    o = _setup(pm, tables, mats, hu, vox)
    spot = inputs.plan_single_spot((2.1, 2.1, 0.0), 140.0, 0.3)
    dg, sg, do, so, cg, co = _dose_parity(pm, o, hu, vox, mats, spot, 400_000, 71, seed_o=72)
    rho = _density(hu, mats)
    assert rho.min() == pytest.approx(0.4) and rho.max() == pytest.approx(1.8)
    for val in (-900, -250, 700, 1500):                                            # energy deposited per HU value
        m = hu == val
        a, b = (dg * rho)[m].sum(), (do * rho)[m].sum()
        assert b > 0 and abs(a / b - 1) < 1e-2, (val, a, b)


def test_call_order_and_argument_errors(tables):
    from paper_1409_8336_b200 import Pmc, PmcError
    p = Pmc(0)
    w = inputs.workload("c1")
    with pytest.raises(PmcError) as e:
        p.set_hu_materials(w["materials"])
    assert e.value.code == -2                                             # PMC_E_STATE
    p.load_physics_tables(tables)
    p.shape = w["hu"].shape
    with pytest.raises(PmcError) as e:
        p.simulate(w["spots"], 10, 1)
    assert e.value.code == -2
    p.set_hu_materials(w["materials"])
    with pytest.raises(PmcError):
        p.load_ct(w["hu"], (0.2, -0.2, 0.2))
    with pytest.raises(PmcError):
        p.set_option("no_such_option", 1.0)
    mats = [dict(m) for m in w["materials"]]
    mats[1] = dict(mats[1], hu_lo=mats[1]["hu_lo"] + 1)
    with pytest.raises(PmcError):
        p.set_hu_materials(mats)
    p.close()


def test_scratch_comes_from_the_callers_allocator(tables):
    """pmc_create_with_allocator: with the binding's default the queues and tallies are PyTorch allocations
    (torch sees them, and they return to its pool when the context is destroyed); with torch_allocator=False they are
    plain cudaMalloc and torch sees nothing.  Same result either way."""
    from paper_1409_8336_b200 import Pmc
    w = inputs.workload("c1")
    hu = torch.as_tensor(w["hu"], device="cuda")
    doses = []
    import gc
    for use_torch in (True, False):
        # garbage of earlier tests (contexts, result tensors in reference cycles) must be gone BEFORE the baseline is read:
        # if the collector frees it in the middle of this test the torch-side byte count drops and the deltas below lie
        gc.collect()
        torch.cuda.synchronize(); torch.cuda.empty_cache()
        before = torch.cuda.memory_allocated()
        p = Pmc(0, torch_allocator=use_torch)
        p.load_physics_tables(tables); p.set_hu_materials(w["materials"]); p.load_ct(hu, w["vox"])
        d, _ = p.simulate(w["spots"], 20_000, 5)
        doses.append(d.clone())
        held = torch.cuda.memory_allocated() - before - 3 * d.numel() * 4          # minus dose, sigma and the clone
        # six queues of 12 words x 1.25 x 20000 histories + 10 tallies of 250000 voxels = about 17 MB
        assert (held > 12e6) if use_torch else (abs(held) < 1e6), (use_torch, held)
        p.close(); del d
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() - before < 4e6                      # only the result tensors are left
    assert torch.equal(doses[0], doses[1]) or torch.allclose(doses[0], doses[1], rtol=2e-4, atol=1e-16)


def test_streams_are_schedule_independent(pm, tables):
    """Philox streams are keyed per history (north_star): sub-group size, history offset and the stream the context
    runs on change the schedule, not the physics.  Integer counters are identical; float tallies agree up to the
    order of the atomic adds."""
    w = inputs.workload("c1")
    _setup(pm, tables, w["materials"], w["hu"], w["vox"])
    n = 30_000
    d0, _ = pm.simulate(w["spots"], n, 77); c0 = pm.counters()
    pm.set_option("chunk_histories", 1000.0)
    d1, _ = pm.simulate(w["spots"], n, 77); c1 = pm.counters()
    pm.set_option("chunk_histories", float(1 << 21))
    pm.set_option("dose_aggregate", 1.0)                                  # warp-merged atomics (default: plain RED)
    d2, _ = pm.simulate(w["spots"], n, 77); c2 = pm.counters()
    pm.set_option("dose_aggregate", 0.0)
    for c in (c1, c2):
        for k in ("n_steps", "n_elastic", "n_nonelastic", "n_secondary_protons", "n_inc_tries"):
            assert c[k] == c0[k], k
    for d in (d1, d2):
        assert torch.allclose(d, d0, rtol=2e-4, atol=1e-16)
    # two halves with history offsets = the whole (sharding)
    pm.set_option("n_batches", 2.0)
    dw, _ = pm.simulate(w["spots"], n, 78); cw = pm.counters()
    pm.set_option("n_batches", 10.0)
    da, _ = pm.simulate(w["spots"], n // 2, 78); ca = pm.counters()
    pm.set_option("history_offset", float(n // 2))
    db, _ = pm.simulate(w["spots"], n // 2, 78); cb = pm.counters()
    pm.set_option("history_offset", 0.0)
    assert ca["n_steps"] + cb["n_steps"] == cw["n_steps"] and ca["n_nonelastic"] + cb["n_nonelastic"] == cw["n_nonelastic"]
    assert torch.allclose(0.5 * (da + db), dw, rtol=2e-4, atol=1e-16)
