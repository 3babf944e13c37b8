"""More pins of the fp64 CPU oracle (CPU only, `-m "not gpu"`): the functions VERDICT r01 listed as unpinned.

NN angular law and Cugnon values, shell-boundary refraction/reflection, Pauli blocking and the trapping rule, the
discrete-event rate and its elastic / non-elastic / element branching, the multi-spot sampler with divergence, and the
cascade step guard.  As in test_oracle_pins.py the expected values never come from the oracle: they are the numbers of
SURVEY 8(c).6 (the reading of PAPER.md:L77 ref [20]), closed forms of classical mechanics and of the exponential
attenuation law, or exact inequalities.  Each docstring names the deliberate break that makes the test fail.
"""
import numpy as np
import pytest
from scipy import stats

import inputs
from inputs.physics_tables import M_P
from oracle import Oracle, philox4x32_10
from oracle import binding as ob

M_N = 939.56542052
N_AVO = 6.02214076e23


# ------------------------------------------------------------------ Cugnon values (PAPER.md:L77 ref [20])
def test_cugnon_joint_values_of_the_survey():
    """sigma_pp / sigma_np at every joint, from below and from above, against the values SURVEY 8(c).6 prints
    (pp 27.8/28.1 @0.44, 23.60/23.61 @0.8, 22.08/22.00 @2; np 68.4/68.3 @0.446, 34.71/34.66 @0.8).  A wrong coefficient
    or exponent in any segment moves one of its two end values (breaks when e.g. -2.104 -> -2.0 or 1250 -> 1200)."""
    eps = 1e-9
    for which, p, lo, hi, tol in [(0, 0.44, 27.8, 28.1, 0.06), (0, 0.8, 23.60, 23.61, 0.006), (0, 2.0, 22.08, 22.00, 0.006),
                                  (1, 0.446, 68.4, 68.3, 0.06), (1, 0.8, 34.71, 34.66, 0.006)]:
        assert ob.cugnon(which, p * (1 - eps)) == pytest.approx(lo, abs=tol), (which, p)
        assert ob.cugnon(which, p * (1 + eps)) == pytest.approx(hi, abs=tol), (which, p)


def test_cugnon_segment_interiors():
    """Inside the segments: the SURVEY formulas typed out here, at momenta away from the joints (T_lab 50-250 MeV is
    p_lab 0.310-0.729 GeV/c).  Also B_pp, B_np and a(p), which no joint test looks at."""
    pp = lambda p: (34.0 * (p / 0.4) ** -2.104 if p < 0.44 else 23.5 + 1000 * (p - 0.7) ** 4 if p < 0.8 else
                    1250 / (p + 50) - 4 * (p - 1.3) ** 2 if p < 2 else 77 / (p + 1.5))
    np_ = lambda p: (6.3555 * p ** -3.2481 * np.exp(-0.377 * np.log(p) ** 2) if p < 0.446 else
                     33 + 196 * abs(p - 0.95) ** 2.5 if p < 0.8 else 31 / np.sqrt(p) if p < 2 else 77 / (p + 1.5))
    bpp = lambda p: 5.5 * p ** 8 / (7.7 + p ** 8)
    bnp = lambda p: 0.0 if p < 0.225 else 16.53 * (p - 0.225) if p < 0.6 else -1.63 * p + 7.16 if p < 1.6 else bpp(p)
    anp = lambda p: 1.0 if p < 0.8 else 0.64 / p ** 2
    for p in (0.2, 0.31, 0.4, 0.5, 0.62, 0.729, 0.9, 1.3, 1.7, 1.9, 2.5):
        assert ob.cugnon(0, p) == pytest.approx(pp(p), rel=1e-12)
        assert ob.cugnon(1, p) == pytest.approx(np_(p), rel=1e-12)
        assert ob.cugnon(4, p) == pytest.approx(anp(p), rel=1e-12)
        if p < 2:         # SURVEY gives B only below 2 GeV/c (T_lab < 1.27 GeV; the method stops at 250 MeV)
            assert ob.cugnon(2, p) == pytest.approx(bpp(p), rel=1e-12)
            assert ob.cugnon(3, p) == pytest.approx(bnp(p), rel=1e-12, abs=1e-15)
    # hand-computed anchors (not via the lambdas above): 34 x 0.75^-2.104 = 62.28 mb; 31/sqrt(1.21) = 28.18 mb
    assert ob.cugnon(0, 0.3) == pytest.approx(62.28, abs=0.02) and ob.cugnon(1, 1.21) == pytest.approx(28.18, abs=0.01)
    assert ob.cugnon(3, 0.5) == pytest.approx(4.546, abs=1e-3) and ob.cugnon(3, 1.0) == pytest.approx(5.53, abs=1e-9)


# ------------------------------------------------------------------ NN angular law (Reading R6.6)
def _g(t, B, tmax):
    """CDF of |t| ~ exp(-B |t|) on [0, tmax]"""
    t = np.clip(t, 0.0, tmax)
    return t / tmax if B * tmax < 1e-12 else (1 - np.exp(-B * t)) / (1 - np.exp(-B * tmax))


def _pcm(t_lab, m_proj, m_targ):
    plab = np.sqrt(t_lab * (t_lab + 2 * m_proj))
    s = m_proj ** 2 + m_targ ** 2 + 2 * m_targ * (t_lab + m_proj)
    return plab, m_targ * plab / np.sqrt(s)


@pytest.mark.parametrize("same,p_gev,B,a", [
    (True, 1.5, 5.5 * 1.5 ** 8 / (7.7 + 1.5 ** 8), 0.0),       # pp: exp(B t) only
    (True, 0.644, 5.5 * 0.644 ** 8 / (7.7 + 0.644 ** 8), 0.0),
    (False, 0.2, 0.0, 1.0),                                      # np below 0.225 GeV/c: isotropic
    (False, 0.5, 16.53 * (0.5 - 0.225), 1.0),                   # np: exp(B t) + a exp(B u), a = 1
    (False, 1.0, -1.63 * 1.0 + 7.16, 0.64),                     # a = 0.64 / p^2
    (False, 1.3, -1.63 * 1.3 + 7.16, 0.64 / 1.69)])
def test_nn_angular_law_against_analytic_cdf(same, p_gev, B, a):
    """cos(theta_cm) of sample_nn_cos against the analytic CDF of e^{Bt} (+ a e^{Bu}) on [0, 4 p_cm^2], with B and a typed
    from SURVEY 8(c).6 item 6, and the backward fraction a/(1+a).  Fails if B_pp/B_np are swapped or unused (isotropic), if
    the backward branch has the wrong sign or weight (a vs 1/a), or if t is not truncated at 4 p_cm^2."""
    n = 200_000
    plab = p_gev * 1e3
    t_lab = np.sqrt(plab ** 2 + M_P ** 2) - M_P
    _, pcm = _pcm(t_lab, M_P, M_P if same else M_N)
    tmax = 4 * pcm * pcm * 1e-6
    c = ob.nn_cos(same, p_gev, pcm, n, 77)
    assert np.all(np.abs(c) <= 1.0)

    def cdf(x):           # forward branch: cos = 1 - 2t/tmax; backward: cos -> -cos
        fwd = 1 - _g(tmax * (1 - x) / 2, B, tmax)
        bwd = _g(tmax * (1 + x) / 2, B, tmax)
        return (fwd + a * bwd) / (1 + a)

    assert stats.kstest(c, cdf).pvalue > 1e-3
    if not same and B * tmax > 3:      # the two lobes are separated: the backward one holds a/(1+a) of the events
        want = (a * _g(tmax / 2, B, tmax) + (1 - _g(tmax / 2, B, tmax))) / (1 + a)
        assert abs(np.mean(c < 0) - want) < 4.5 * np.sqrt(want * (1 - want) / n)
        assert np.mean(c < 0) == pytest.approx(a / (1 + a), abs=0.03)


@pytest.mark.parametrize("target,t_in", [("n", 150.0), ("n", 400.0), ("p", 800.0)])
def test_cascade_collisions_follow_the_angular_law(target, t_in):
    """The law as the cascade uses it: a dilute one-shell 'nucleus' of nucleons at rest (p_F = 0, V = 0, Pauli off, constant
    tiny cross-section, so at most one collision matters).  Attempts that put exactly two nucleons out had exactly one
    collision; the struck nucleon's kinetic energy gives the invariant |t| = 2 m T_recoil, which must follow
    e^{Bt} (+ a e^{Bu}) at the projectile's lab momentum.  Fails if inc_attempt passes the wrong 'same type' flag, the CM
    instead of the lab momentum, or scatters about the wrong axis (the recoil energy would not match |t|)."""
    R, rho, sig = 4.0, 0.1, 0.5                                  # lambda = 1/(rho sigma 0.1 fm2/mb) = 200 fm >> R
    col = 0 if target == "p" else 1
    dens = np.zeros((2, 1)); dens[col, 0] = rho
    n = 1_500_000
    n_out, rec = ob.inc_custom([R], dens, np.zeros((2, 1)), np.zeros((2, 1)), t_in, n, 5, const_sigma_mb=sig)
    two = np.abs(np.where(n_out < 0, -1 - n_out, n_out)) == 2
    assert two.sum() > 8000
    ke = rec[two][:, :2, 1]; ty = rec[two][:, :2, 0]
    assert np.allclose(ke.sum(axis=1), t_in, atol=1e-9)          # elastic, V = 0: kinetic energy is shared
    m_t = M_P if target == "p" else M_N
    plab, pcm = _pcm(t_in, M_P, m_t)
    tmax = 4 * pcm * pcm * 1e-6
    p = plab * 1e-3
    if target == "n":
        assert np.all(np.sort(ty, axis=1) == [0, 1])
        t_rec = np.where(ty[:, 0] == 1, ke[:, 0], ke[:, 1])      # the neutron is the struck one
        B = 0.0 if p < 0.225 else 16.53 * (p - 0.225) if p < 0.6 else -1.63 * p + 7.16
        a = 1.0 if p < 0.8 else 0.64 / p ** 2
        t = 2 * m_t * t_rec * 1e-6
        cdf = lambda x: (_g(x, B, tmax) + a * (1 - _g(tmax - x, B, tmax))) / (1 + a)
    else:
        assert np.all(ty == 0)
        B = 5.5 * p ** 8 / (7.7 + p ** 8)
        t = 2 * m_t * ke.min(axis=1) * 1e-6                       # identical particles: the smaller of |t| and |u|
        cdf = lambda x: _g(x, B, tmax) + 1 - _g(tmax - x, B, tmax)
        assert B * tmax > 2                                       # far from isotropic at this momentum
    assert t.max() <= tmax * (1 + 1e-9)
    # (a second collision, probability ~ R / lambda = 2 %, would have put a third nucleon out: excluded above)
    assert stats.kstest(t, cdf).pvalue > 1e-3


# ------------------------------------------------------------------ shell boundaries ("reflection and refraction"; Reading R6.5)
def _sweep_deflection(b, p0, shells):
    """Classical scattering angle of a particle with impact parameter b and asymptotic momentum p0 in a piecewise-constant
    central potential: angular momentum L = b p0 is conserved, inside a shell of momentum p the path is a straight chord at
    distance L/p from the centre, and the polar angle swept between radii ra < rb on that chord is acos(d/rb) - acos(d/ra).
    shells = [(r_outer, p_inside)] from the outside in.  Returns cos(Theta)."""
    L = b * p0
    r_out = shells[0][0]
    sweep = np.arcsin(b / r_out)                                  # free flight from infinity to the surface
    for k, (rb, p) in enumerate(shells):
        d = L / p
        if d >= rb:                                               # cannot enter this shell: reflected at rb
            break
        ra = shells[k + 1][0] if k + 1 < len(shells) else 0.0
        if d >= ra:                                               # turning point of the chord inside this shell
            sweep += np.arccos(d / rb)
            break
        sweep += np.arccos(d / rb) - np.arccos(d / ra)
    return np.cos(np.pi - 2 * sweep)


@pytest.mark.parametrize("radii,depth", [
    ([5.0], [40.0]),                        # one attractive well: two refractions
    ([2.5, 5.0], [60.0, 25.0]),             # deeper inside: four refractions (inward and outward crossings)
    ([3.0, 5.0], [-30.0, 35.0]),            # repulsive core: refraction or total reflection at the inner boundary
    ([2.0, 3.5, 5.0], [10.0, 45.0, 20.0])])
def test_shell_boundaries_conserve_energy_and_angular_momentum(radii, depth):
    """No collisions (zero density): the proton only meets shell boundaries.  It must leave with exactly its incident
    kinetic energy (eps = T - V conserved at every crossing) and deflected by the classical scattering angle of the
    piecewise-constant potential, which follows from conservation of angular momentum, i.e. of the tangential momentum at
    each boundary; reflection happens exactly when the chord cannot enter.  The impact parameter of attempt i is
    r_max sqrt(u), u the first draw of stream (seed, i).  Fails if the tangential momentum is not kept, if p_r^2 < 0 does not
    reflect, if the entry refraction is skipped, or if T' = T + (V_new - V_old) has the wrong sign."""
    ns = len(radii); n = 4000; seed = 9; t_in = 150.0
    V = np.array([depth, depth], dtype=float)                    # shell 0 is the innermost
    n_out, rec = ob.inc_custom(radii, np.zeros((2, ns)), np.zeros((2, ns)), V, t_in, n, seed)
    assert np.all(n_out == -2)                                    # one nucleon out, attempt rejected (no collision)
    assert np.all(rec[:, 0, 0] == 0) and np.allclose(rec[:, 0, 1], t_in, atol=1e-9)
    u0 = np.array([(philox4x32_10([i, 0, 0, 0], [seed, 0])[0] + 0.5) / 2.0 ** 32 for i in range(n)])
    b = radii[-1] * np.sqrt(u0)
    mom = lambda t: np.sqrt(t * (t + 2 * M_P)) if t > 0 else 0.0
    shells = [(radii[k], mom(t_in + depth[k])) for k in range(ns - 1, -1, -1)]
    want = np.array([_sweep_deflection(bb, mom(t_in), shells) for bb in b])
    assert np.max(np.abs(rec[:, 0, 4] - want)) < 1e-9
    assert np.allclose(np.linalg.norm(rec[:, 0, 2:5], axis=1), 1.0, atol=1e-12)
    # the deflection lies in the plane of incidence: the outgoing direction has no component along z x r_entry
    u1 = np.array([(philox4x32_10([i, 0, 0, 0], [seed, 0])[1] + 0.5) / 2.0 ** 32 for i in range(n)])
    phi = 2 * np.pi * u1
    assert np.max(np.abs(-rec[:, 0, 2] * np.sin(phi) + rec[:, 0, 3] * np.cos(phi))) < 1e-9
    if min(depth) < 0:                                            # the repulsive core does reflect some and transmit others
        core = [(radii[0], mom(t_in + depth[0]))]
        inner_d = b * mom(t_in) / core[0][1]
        reach = b * mom(t_in) / shells[-2][1] < radii[0]
        assert np.any(reach & (inner_d >= radii[0])) and np.any(inner_d < radii[0])


# ------------------------------------------------------------------ Pauli blocking and trapping (Reading R6.4)
def test_pauli_blocking_in_a_one_shell_fermi_gas():
    """One dilute shell of neutrons with p_F = 250 MeV/c and V = 0: with Pauli blocking on, both products of every accepted
    collision are above their Fermi energy (neutron 32.7 MeV, proton 0), so no struck neutron leaves below 32.7 MeV; with
    blocking off the same streams give more collisions and many soft neutrons.  Fails if the Pauli test is dropped, applied
    to one product only, or compares with the other type's Fermi energy."""
    R, rho, pf, t_in, n = 4.0, 0.1, 250.0, 100.0, 600_000
    ef_n = np.sqrt(pf ** 2 + M_N ** 2) - M_N
    assert ef_n == pytest.approx(32.7, abs=0.1)
    dens = np.array([[0.0], [rho]]); pF = np.array([[0.0], [pf]])
    cnt = {}
    for pauli in (True, False):
        n_out, rec = ob.inc_custom([R], dens, pF, np.zeros((2, 1)), t_in, n, 3, pauli=pauli, const_sigma_mb=2.0)
        k = np.where(n_out < 0, -1 - n_out, n_out)
        two = k == 2
        ke, ty = rec[two][:, :2, 1], rec[two][:, :2, 0]
        kn = np.where(ty[:, 0] == 1, ke[:, 0], ke[:, 1])
        cnt[pauli] = (int((k >= 2).sum()), float(np.mean(kn < ef_n)), float(kn.min()))
    assert cnt[True][0] > 3000 and cnt[True][1] == 0.0 and cnt[True][2] > ef_n
    assert cnt[False][0] > 1.15 * cnt[True][0] and cnt[False][1] > 0.1


@pytest.mark.parametrize("Z,A,e_mev", [(8, 16, 150.0), (22, 48, 230.0), (20, 40, 70.0)])
def test_trapping_rule_on_emitted_cascade_nucleons(oracle_c1, Z, A, e_mev):
    """A cascade nucleon whose outside energy eps = T - V is at most B_C = 1.44 (Z-1)/r_max (protons; 0 for neutrons) stays
    in the nucleus, and eps is conserved up to the surface: every INC proton is emitted above B_C, every INC neutron above
    0, with r_max = 1.07 A^(1/3) + 0.545 ln 99 (Reading R6.1).  Fails if the trapping test is dropped (soft protons
    appear: they are the most numerous ones) or uses the neutron's barrier for protons."""
    sec, off = oracle_c1.nonelastic(Z, A, e_mev, 20000, 123)
    rmax = 1.07 * A ** (1 / 3) + 0.545 * np.log(99.0)
    bc = 1.44 * (Z - 1) / rmax
    inc = sec[sec["origin"] == 0]
    p, nn = inc[inc["Z"] == 1], inc[inc["Z"] == 0]
    assert len(p) > 10000 and len(nn) > 3000
    assert p["ke"].min() > bc and nn["ke"].min() > 0.0
    # the cut is sharp, not a property of the spectrum: protons do come out right above B_C, neutrons right above 0
    assert p["ke"].min() < bc + 1.0 and nn["ke"].min() < 0.5
    assert 1.5 < bc < 6.5


# ------------------------------------------------------------------ event rate and branching (Reading R3.1, R5)
def _slab_expectation(tables, mat, hu, e0, thick, o):
    """Expected events per primary, per class and element, in a slab: the exponential attenuation law with the
    macroscopic cross-sections n_i sigma_i built here from the input tables (n_i = rho N_A w_i / A_i), sigma linear in
    ln E, the energy along the depth from the (separately pinned) range tables.  A primary is removed by a non-elastic
    event or by p-p scattering (which sends both protons below the test's energy cut most of the time)."""
    rho = mat["rho_lo"] + (mat["rho_hi"] - mat["rho_lo"]) * (hu - mat["hu_lo"]) / (mat["hu_hi"] - mat["hu_lo"])
    lne = np.linspace(np.log(tables["e_min"]), np.log(tables["e_max"]), tables["n_e"])
    xs = (np.arange(2000) + 0.5) * thick / 2000
    wf = rho * mat["f_m"] if mat["table_id"] == 0 else rho
    e_x = np.array([o.energy_of_range(mat["table_id"], o.range_gcm2(mat["table_id"], e0) - x * wf) for x in xs])
    nel = len(tables["elem_a"])
    mu = np.zeros((2, nel, xs.size))
    for i in range(nel):
        n_i = rho * N_AVO * mat["w"][i] / tables["elem_a"][i] * 1e-27
        mu[0, i] = n_i * np.interp(np.log(e_x), lne, tables["sigma_el_mb"][i])
        mu[1, i] = n_i * np.interp(np.log(e_x), lne, tables["sigma_ne_mb"][i])
    h = [i for i in range(nel) if tables["elem_a"][i] == 1]
    removing = mu[1].sum(axis=0) + mu[0][h].sum(axis=0)
    dx = thick / xs.size
    surv = np.exp(-(np.cumsum(removing) - 0.5 * removing) * dx)
    return (mu * surv).sum(axis=2) * dx, mu.sum(axis=(0, 1)).mean() * thick


@pytest.mark.parametrize("medium", ["water", "bone"])
def test_event_rate_and_branching_in_a_thin_slab(tables, medium):
    """One homogeneous voxel 0.6 cm thick, MCS and straggling off, 150 MeV.  (i) events per primary = 1 - exp(-Sigma L)
    with Sigma = sum n_i (sigma_el,i + sigma_ne,i) from the tables; (ii) elastic / non-elastic and the target element are
    chosen in proportion to n_i sigma_i (chi^2 over the classes x elements).  The energy cut is raised to 120 MeV so that
    secondaries end where they are born and the counts are those of the primaries.  Fails with n_i off by a factor, lambda
    sampled from the wrong Sigma, sigma_el and sigma_ne swapped, or element weights ~ w_i instead of n_i sigma_i."""
    t = dict(tables); t["e_cut"] = 120.0
    if medium == "water":
        mats, hu = inputs.make_materials_c1(), 0
    else:
        mats, hu = inputs.make_materials_24(), 1200
    mat = [m for m in mats if m["hu_lo"] <= hu < m["hu_hi"]][0]
    thick, e0, n = 0.6, 150.0, 3_000_000
    o = Oracle(t, mats)
    o.load_ct(np.full((1, 1, 1), hu, dtype=np.int16), (50.0, 50.0, thick))
    for k in ("straggling", "mcs"):
        o.set_option(k, 0)
    o.simulate(inputs.plan_single_spot((25.0, 25.0, 0.0), e0, 0.0), n, 17)
    el, ne = o.event_counts()
    c = o.counters()
    assert el.sum() == c["n_elastic"] and ne.sum() == c["n_nonelastic"]
    want, sigma_l = _slab_expectation(t, mat, hu, e0, thick, o)
    got = np.stack([el, ne])[:, :want.shape[1]].astype(float)
    tot_w, tot_g = want.sum() * n, got.sum()
    assert 0.005 < sigma_l < 0.05
    # (i) rate: 4 sigma of the Poisson count + 0.7 % for the second-order terms (a scattered primary's later events)
    assert abs(tot_g / tot_w - 1) < 4 / np.sqrt(tot_w) + 7e-3, (tot_g, tot_w)
    assert tot_g / n == pytest.approx(1 - np.exp(-sigma_l), rel=0.03)
    # (ii) branching: chi^2 of the class x element table against n_i sigma_i / Sigma
    m = want > 0
    assert np.all(got[~m] == 0) and m.sum() >= 3
    exp_counts = want[m] / want[m].sum() * tot_g
    chi2 = ((got[m] - exp_counts) ** 2 / exp_counts).sum()
    assert stats.chi2.sf(chi2, m.sum() - 1) > 1e-4, (got[m], exp_counts)
    # and the split by class alone
    assert got[0].sum() / tot_g == pytest.approx(want[0].sum() / want.sum(), abs=4 * np.sqrt(0.25 / tot_g) + 2e-3)


# ------------------------------------------------------------------ multi-spot sampler with divergence (Reading R2)
def test_spot_frequencies_and_divergence(tables):
    """Five spots of unequal weight (one of them zero), different positions, sizes, divergences and axes: chi^2 of the spot
    frequencies against the normalised weights; per spot the sample sigma of position and of the direction cosines equals
    sigma_x/sigma_y and div_x/div_y in the spot's own transverse frame.  Fails if the CDF lookup is off by one spot, if
    weights are not normalised, if x and y are swapped, or if the divergence branch uses the position deviates."""
    o = Oracle(tables, inputs.make_materials_c1())
    o.load_ct(np.zeros((1, 1, 1), dtype=np.int16), (400.0, 400.0, 400.0))
    mk = inputs.plan_single_spot
    spots = np.concatenate([
        mk((100.0, 100.0, 50.0), 100.0, 0.3), mk((150.0, 120.0, 50.0), 120.0, 0.5),
        mk((200.0, 200.0, 50.0), 140.0, 0.4), mk((250.0, 260.0, 50.0), 160.0, 0.2),
        mk((50.0, 300.0, 200.0), 180.0, 0.6, direction=(1.0, 0.0, 0.0))])
    w = np.array([1.0, 3.5, 0.0, 0.25, 2.0]); spots[:, 12] = w
    sx = np.array([0.3, 0.5, 0.4, 0.2, 0.6]); sy = np.array([0.45, 0.25, 0.4, 0.3, 0.15])
    dvx = np.array([0.004, 0.0, 0.01, 0.002, 0.008]); dvy = np.array([0.001, 0.006, 0.01, 0.0, 0.003])
    spots[:, 8], spots[:, 9], spots[:, 10], spots[:, 11] = sx, sy, dvx, dvy
    n = 400_000
    s = o.sample_primaries(spots, n, 21)
    idx = s[:, 0].astype(int)
    assert np.all(idx >= 0)
    cnt = np.bincount(idx, minlength=5)
    assert cnt[2] == 0
    m = w > 0
    exp_counts = w[m] / w.sum() * n
    assert stats.chi2.sf(((cnt[m] - exp_counts) ** 2 / exp_counts).sum(), m.sum() - 1) > 1e-4, cnt
    for k in (0, 1, 3, 4):
        q = s[idx == k]; se = 4.5 / np.sqrt(2 * len(q))
        # transverse frame of Reading R2: axis +z -> (ex, ey) = (x, y); axis +x -> (ex, ey) = (y, z)
        pa, pb, da, db = (q[:, 1], q[:, 2], q[:, 4], q[:, 5]) if k != 4 else (q[:, 2], q[:, 3], q[:, 5], q[:, 6])
        assert pa.std() == pytest.approx(sx[k], rel=se) and pb.std() == pytest.approx(sy[k], rel=se)
        assert pa.mean() == pytest.approx(spots[k, 0 if k != 4 else 1], abs=4.5 * sx[k] / np.sqrt(len(q)))
        for d, dv in ((da, dvx[k]), (db, dvy[k])):
            if dv > 0:
                assert d.std() == pytest.approx(dv, rel=se + 1e-4)
            elif dvx[k] == 0 and dvy[k] == 0:
                assert np.all(d == 0)
            else:
                assert d.std() < 1e-12
        assert np.allclose(np.linalg.norm(q[:, 4:7], axis=1), 1.0, atol=1e-12)
        assert np.all(q[:, 7] == spots[k, 6])
        assert abs(np.corrcoef(pa, da)[0, 1]) < 5 / np.sqrt(len(q)) if dvx[k] > 0 else True


# ------------------------------------------------------------------ the cascade step guard (Reading R6.8)
def test_cascade_step_guard_is_harmless(oracle_c1):
    """Reading R6.8 abandons a cascade attempt after 1024 tracking steps (the paper has no limit).  On the
    heaviest target and highest energy of the configs (p + 48Ti at 230 MeV): the guard trips in fewer than 1e-5 of the
    attempts, the same streams with guard 20000 give the same events when it never trips, and the 200-nucleon stack limit is
    never reached; the deepest stack and the most nucleons out are far below the CUDA path's fixed capacities (48 and 32).
    With a guard of 30 steps the yields do change - the test can see a guard that bites."""
    o = oracle_c1
    n = 150_000
    res = {}
    try:
        for guard in (1024, 20000, 30):
            o.set_option("inc_step_guard", guard)
            sec, off = o.nonelastic(22, 48, 230.0, n if guard != 30 else 30000, 4242)
            res[guard] = (sec, off, o.counters())
    finally:
        o.set_option("inc_step_guard", 1024)
    c0, c1 = res[1024][2], res[20000][2]
    assert c0["n_inc_guard_trips"] <= 1e-5 * c0["n_inc_tries"] and c1["n_inc_guard_trips"] == 0
    assert c0["n_inc_stack_trips"] == 0 and c1["n_inc_stack_trips"] == 0
    assert c0["inc_max_stack"] <= 16 and c0["inc_max_out"] <= 16
    if c0["n_inc_guard_trips"] == 0:
        assert np.array_equal(res[1024][1], res[20000][1]) and res[1024][0].tobytes() == res[20000][0].tobytes()
    else:
        for zz, aa in ((0, 1), (1, 1), (2, 4)):
            ya = np.sum((res[1024][0]["Z"] == zz) & (res[1024][0]["A"] == aa)) / n
            yb = np.sum((res[20000][0]["Z"] == zz) & (res[20000][0]["A"] == aa)) / n
            assert abs(ya - yb) < 3 * np.sqrt((ya + yb) / n)
    cb = res[30][2]
    assert cb["n_inc_guard_trips"] > 0.01 * cb["n_inc_tries"]
