"""Pins for the fp64 oracle: closed forms, the value the paper prints for eq. (23), invariants and
brute force through independent scipy routines.  CPU only."""
import math
import os

import numpy as np
import pytest
from scipy import integrate, optimize, special

import oracle as O
from workloads import append_pixels, lambda_vector, make_workload, split_into_pixels

C = 299792.458
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def lam(**kw):
    return lambda_vector(**kw)


# ------------------------------------------------------------------ P1: GR limits of eq. (2)
@pytest.mark.parametrize("kw", [dict(Xi0=1.0, n=0.7), dict(Xi0=1.0, n=4.2), dict(Xi0=0.4, n=0.0),
                                dict(Xi0=3.0, n=0.0)])
def test_p1_xi0_one_or_n_zero_is_gr(kw):
    z = np.linspace(0.0, 6.0, 41)
    d = O.distances(lam(**kw), z)
    assert np.allclose(d["dl_gw"], d["dl_em"], rtol=1e-15, atol=0)


def test_p1_xi_limits():
    # Xi(0) = 1 and Xi(z->inf) = Xi0  (eq. 2): d_L^gw/d_L^em at small and huge z
    la = lam(Xi0=1.8, n=2.5)
    d = O.distances(la, np.array([1e-9, 9.9]))
    r = d["dl_gw"] / d["dl_em"]
    assert abs(r[0] - 1.0) < 1e-8
    assert abs(r[1] - (1.8 + (1 - 1.8) / 10.9 ** 2.5)) < 1e-14


# ------------------------------------------------------------------ P2: closed-form cosmologies
def test_p2_einstein_de_sitter():
    z = np.array([0.01, 0.3, 1.0, 2.5, 8.0])
    d = O.distances(lam(Om=1.0, H0=67.0), z)
    ref = (1 + z) * (2 * C / 67.0) * (1 - 1 / np.sqrt(1 + z))
    assert np.allclose(d["dl_em"], ref, rtol=1e-13)


def test_p2_empty_limit_and_inverse():
    la = lam(Om=1e-15, H0=70.0, Xi0=1.0)
    z = np.array([0.05, 0.7, 3.0])
    d = O.distances(la, z)
    assert np.allclose(d["dc"], C * z / 70.0, rtol=1e-12)
    dl = np.array([300.0, 5000.0, 40000.0])
    zi = O.z_of_dl(la, dl, z_table_max=20.0)
    ref = 0.5 * (-1 + np.sqrt(1 + 4 * dl * 70.0 / C))
    assert np.allclose(zi, ref, rtol=1e-11)


def test_p2_eq23_value_printed_by_paper():
    row = [l for l in open(os.path.join(GOLD, "eq23_rate.txt")) if not l.startswith("#")][0].split()
    R0, zmax, H0, Om, g, k, zp, printed = map(float, row)
    la = lam(H0=H0, Om=Om, gamma=g, kappa=k, z_p=zp)

    def integrand(z):
        dv, _ = O.volume(la, [z])
        return O.psi(la, [z])[0] / (1 + z) * dv[0] / 1e9          # Mpc^3 -> Gpc^3
    val, _ = integrate.quad(integrand, 0.0, zmax, epsabs=0, epsrel=1e-10)
    rate = R0 * val
    assert float(f"{rate:.1e}") == printed, rate                  # rounds to 1.4e4
    assert abs(rate - 1.366e4) < 0.01e4                           # SURVEY probe value (full sky)


def test_p2_volume_consistency():
    # dVc/dz is the derivative of Vc, and Vc = 4pi/3 dC^3
    la = lam()
    z = np.array([0.2, 0.9, 1.5])
    dv, vc = O.volume(la, z)
    e = 1e-5
    _, vp = O.volume(la, z + e)
    _, vm = O.volume(la, z - e)
    assert np.allclose(dv, (vp - vm) / (2 * e), rtol=1e-8)
    assert np.allclose(vc, 4 * np.pi / 3 * O.distances(la, z)["dc"] ** 3, rtol=1e-14)


# ------------------------------------------------------------------ P3: derivative, round trip
@pytest.mark.parametrize("kw", [dict(), dict(Xi0=0.5, n=3.0, H0=80, Om=0.4), dict(Xi0=2.0, n=0.5, H0=60, Om=0.2)])
def test_p3_derivative_and_round_trip(kw):
    la = lam(**kw)
    z = np.array([0.02, 0.4, 1.3, 4.0])
    e = 1e-5
    f = lambda x: O.distances(la, x)["dl_gw"]
    fd = (f(z + e) - f(z - e)) / (2 * e)
    assert np.allclose(O.distances(la, z)["ddl_gw_dz"], fd, rtol=1e-8)
    assert np.allclose(O.z_of_dl(la, f(z)), z, rtol=0, atol=2e-13)
    assert O.dl_monotone(la)


def test_p3_dc_against_adaptive_quadrature():
    la = lam(H0=73.0, Om=0.31)
    for z in (0.1, 1.0, 3.3, 9.0):
        ref, _ = integrate.quad(lambda x: C / 73.0 / math.sqrt(0.31 * (1 + x) ** 3 + 0.69), 0, z, epsabs=0, epsrel=1e-13)
        assert abs(O.distances(la, [z])["dc"][0] / ref - 1) < 1e-12


def test_table_range_rule():
    la = lam()
    dmax = O.distances(la, [2.0])["dl_gw"][0]
    z = O.z_of_dl(la, [dmax * 0.999, dmax * 1.001], z_table_max=2.0)
    assert np.isfinite(z[0]) and np.isnan(z[1])


def test_nonmonotone_detected():
    # Xi0 << 1 with large n makes d_L^gw(z) turn over (R16)
    assert not O.dl_monotone(lam(Xi0=0.01, n=8.0))


# ------------------------------------------------------------------ P4: one-sample KDE
def test_p4_single_sample_is_gaussian():
    zg = np.linspace(0.1, 0.5, 57)
    K = O.kde([0.31], [2.5], 0.02, zg)
    ref = 2.5 * np.exp(-0.5 * ((zg - 0.31) / 0.02) ** 2) / (0.02 * math.sqrt(2 * math.pi))
    assert np.allclose(K, ref, rtol=1e-14)


def test_kde_normalisation_is_by_Ns_not_sum_w():
    # R2: int K dz = mean weight
    rng = np.random.default_rng(1)
    z, w = 0.3 + 0.02 * rng.standard_normal(50), rng.random(50) * 3
    zg = np.linspace(0.0, 0.6, 6001)
    K = O.kde(z, w, 0.004, zg)
    assert abs(np.trapezoid(K, zg) - w.mean()) < 1e-10 * w.mean()


# ------------------------------------------------------------------ P5: closed form of the event integral
def test_p5_event_integral_closed_form():
    rng = np.random.default_rng(2)
    ns, ngal = 40, 7
    z = 0.4 + 0.03 * rng.standard_normal(ns)
    w = rng.random(ns) + 0.1
    h = 0.006
    zgal = 0.4 + 0.04 * rng.standard_normal(ngal)
    sg = 0.0015 * (1 + zgal)
    zg = np.linspace(0.1, 0.7, 1201)                              # dz = 5e-4 <~ sigma_g
    pgal = np.mean(np.exp(-0.5 * ((zg[:, None] - zgal) / sg) ** 2) / (sg * math.sqrt(2 * math.pi)), axis=1)
    K = O.kde(z, w, h, zg)
    I = O.event_integral(lam(), zg, K, pgal)
    s2 = h * h + sg ** 2
    ref = np.mean(w[:, None] * np.mean(np.exp(-0.5 * (z[:, None] - zgal) ** 2 / s2) / np.sqrt(2 * math.pi * s2), axis=1, keepdims=True))
    ref = np.mean(w * np.mean(np.exp(-0.5 * (z[:, None] - zgal[None, :]) ** 2 / s2) / np.sqrt(2 * math.pi * s2), axis=1))
    assert abs(I / ref - 1) < 1e-10


def test_p5_flat_pgal_gives_mean_weight():
    rng = np.random.default_rng(3)
    z, w = 0.5 + 0.01 * rng.standard_normal(30), rng.random(30)
    zg = np.linspace(0.3, 0.7, 2001)
    K = O.kde(z, w, 0.003, zg)
    assert abs(O.event_integral(lam(), zg, K, np.ones_like(zg)) / w.mean() - 1) < 1e-11


def test_trapezoid_on_nonuniform_grid():
    zg = np.array([0.0, 0.1, 0.25, 0.27, 0.6])
    K = np.array([1.0, 2.0, 0.5, 4.0, 1.0])
    p = np.array([2.0, 1.0, 3.0, 0.5, 1.0])
    y = K * p
    ref = sum(0.5 * (y[i] + y[i + 1]) * (zg[i + 1] - zg[i]) for i in range(4))
    assert abs(O.event_integral(lam(), zg, K, p) - ref) < 1e-15


# ------------------------------------------------------------------ P6: mass function
MASS_LAMS = [dict(), dict(alpha=1.0), dict(beta=-1.0), dict(alpha=2.2, beta=0.0, delta_m=9.0, m_low=3.0, m_high=60.0, mu_g=30.0, sigma_g=1.0, lambda_g=0.3),
             dict(delta_m=0.05), dict(m_high=8.0, delta_m=6.0, lambda_g=0.5)]


@pytest.mark.parametrize("kw", MASS_LAMS)
def test_p6_primary_integrates_to_one(kw):
    la = lam(**kw)
    p = dict(zip(("m_low", "delta_m", "m_high", "mu_g", "sigma_g"), (la[7], la[6], la[8], la[9], la[10])))
    pts = sorted({p["m_low"], p["m_low"] + p["delta_m"], p["m_high"], p["mu_g"]})
    top = max(p["m_high"], p["mu_g"] + 30 * p["sigma_g"]) + 1
    tot = 0.0
    edges = [e for e in pts if e < top] + [top]
    for a, b in zip(edges[:-1], edges[1:]):
        v, _ = integrate.quad(lambda m: O.p_m1(la, [m])[0], a, b, epsabs=0, epsrel=1e-11, limit=400)
        tot += v
    assert abs(tot - 1) < 1e-9


@pytest.mark.parametrize("kw", MASS_LAMS)
@pytest.mark.parametrize("frac", [0.04, 0.1, 0.3, 0.95, 1.0, 4.0])
def test_p6_secondary_integrates_to_one(kw, frac):
    la = lam(**kw)
    m_low, dm = la[7], la[6]
    m1 = m_low + frac * dm
    pts = [m_low] + ([m_low + dm] if m1 > m_low + dm else []) + [m1]
    if frac < 0.3:      # deep in the window the integrand piles up at the upper end: help quad find it
        pts = [m_low, m1 - 0.5 * (m1 - m_low), m1 - 0.1 * (m1 - m_low), m1]
    tot = sum(integrate.quad(lambda m: O.p_m2_given_m1(la, [m1], [m])[0], a, b, epsabs=0, epsrel=1e-11, limit=400)[0]
              for a, b in zip(pts[:-1], pts[1:]))
    assert abs(tot - 1) < 1e-9


def test_p6_sharp_limit_is_truncated_power_laws():
    # delta_m -> 0, lambda_g = 0: p(m1) = PL on [m_low, m_high], p(m2|m1) = (b+1) m2^b/(m1^(b+1) - m_low^(b+1))
    a, b, ml, mh = 2.3, 1.4, 5.0, 80.0
    la = lam(alpha=a, beta=b, m_low=ml, m_high=mh, delta_m=1e-9, lambda_g=0.0)
    m1 = np.array([6.0, 20.0, 79.0])
    m2 = np.array([5.5, 11.0, 40.0])
    p1 = (1 - a) * m1 ** (-a) / (mh ** (1 - a) - ml ** (1 - a))
    p2 = (b + 1) * m2 ** b / (m1 ** (b + 1) - ml ** (b + 1))
    assert np.allclose(O.p_m1(la, m1), p1, rtol=1e-8)
    assert np.allclose(O.p_m2_given_m1(la, m1, m2), p2, rtol=1e-8)
    assert np.allclose(O.mass_pdf(la, m1, m2), p1 * p2, rtol=1e-8)


def test_p6_support_and_smoothing_shape():
    la = lam()
    ml, dm, mh = la[7], la[6], la[8]
    m = np.linspace(ml - 1, ml + dm + 1, 400)
    S = O.smoothing(la, m)
    assert np.all(np.diff(S) >= 0) and S[0] == 0 and S[-1] == 1
    assert O.smoothing(la, [ml])[0] == 0 and O.smoothing(la, [ml + dm])[0] == 1
    assert abs(O.smoothing(la, [ml + dm / 2])[0] - 0.5) < 1e-15          # f(dm/2) = 2 - 2 = 0
    # R15 support: m2 < m_low, m2 > m1 -> 0 ; power law is 0 above m_high but the Gaussian is not
    assert O.mass_pdf(la, [30.0], [ml - 0.1])[0] == 0
    assert O.mass_pdf(la, [30.0], [30.1])[0] == 0
    g_only = la[11] * math.exp(-0.5 * ((mh + 1 - la[9]) / la[10]) ** 2) / (la[10] * math.sqrt(2 * math.pi))
    z1 = O.p_m1(la, [40.0])[0] / ((1 - la[11]) * (1 - la[4]) * 40.0 ** -la[4] / (mh ** (1 - la[4]) - ml ** (1 - la[4]))
                                  + la[11] * math.exp(-0.5 * ((40 - la[9]) / la[10]) ** 2) / (la[10] * math.sqrt(2 * math.pi)))
    assert abs(O.p_m1(la, [mh + 1])[0] / (g_only * z1) - 1) < 1e-12


def test_p6_gaussian_component_weight():
    # with S ~ 1 (tiny delta_m) and mu_g well inside, the Gaussian carries exactly lambda_g
    la = lam(delta_m=1e-9, lambda_g=0.25, mu_g=40.0, sigma_g=2.0)
    v, _ = integrate.quad(lambda m: O.p_m1(la, [m])[0], 30.0, 50.0, points=[40.0], epsabs=0, epsrel=1e-12)
    a, ml, mh = la[4], la[7], la[8]
    pl = 0.75 * (50.0 ** (1 - a) - 30.0 ** (1 - a)) / (mh ** (1 - a) - ml ** (1 - a))
    assert abs(v - (pl + 0.25 * special.erf(10 / 2 / math.sqrt(2)))) < 1e-10


# ------------------------------------------------------------------ P7: rate
def test_p7_madau_dickinson():
    la = lam(gamma=2.7, kappa=3.0, z_p=2.0)
    assert abs(O.psi(la, [2.0])[0] - 3.0 ** 2.7 / 2) < 1e-13
    assert abs(O.psi(la, [0.0])[0] - 1 / (1 + 3.0 ** -5.7)) < 1e-15
    lb = lam(gamma=1.9, kappa=2.0, z_p=1e6)
    z = np.array([0.1, 1.0, 3.0])
    assert np.allclose(O.psi(lb, z), (1 + z) ** 1.9, rtol=1e-12)
    # high-z slope is -kappa
    zz = np.array([2000.0, 4000.0])
    p = O.psi(la, zz)
    assert abs(math.log(p[1] / p[0]) / math.log((1 + zz[1]) / (1 + zz[0])) + 3.0) < 1e-6


# ------------------------------------------------------------------ P8: self-consistent injections
def test_p8_unit_weights_give_detected_count():
    w = make_workload("tiny")
    la = w.lam[0]
    n = 500
    dl, m1, m2 = w.inj_dL[:n], w.inj_m1d[:n], w.inj_m2d[:n]
    # p_pop^d(theta_j | lambda*) from the oracle's own pieces -> p_draw := p_pop => s_j = 1
    _, _, s = O.selection_sums(la, dl, m1, m2, np.zeros(n), return_s=True)
    keep = s > 0
    assert keep.sum() > 100
    s1, s2 = O.selection_sums(la, dl[keep], m1[keep], m2[keep], np.log(s[keep]))
    nd, ninj = keep.sum(), 10 * keep.sum()
    assert abs(s1 - nd) < 1e-9 * nd and abs(s2 - nd) < 1e-9 * nd
    assert abs(O.neff(s1, s2, ninj) - nd / (1 - nd / ninj)) < 1e-6


# ------------------------------------------------------------------ P9: xi by quadrature (statistical)
def test_p9_selection_fraction_matches_quadrature():
    la = lam(Xi0=1.3, n=1.5)
    D, zcat = 6000.0, 1.5
    rng = np.random.default_rng(9)
    N = 120_000
    # draw pdf covering the whole support: p(dL) ~ dL^2 on [0, D], m1d ~ 1/m on [4, 400], m2d uniform [4, m1d]
    dl = D * rng.random(N) ** (1.0 / 3.0)
    m1 = 4.0 * (100.0) ** rng.random(N)
    m2 = 4.0 + (m1 - 4.0) * rng.random(N)
    lnp = np.log(3 * dl ** 2 / D ** 3) - np.log(m1 * math.log(100.0)) - np.log(m1 - 4.0)
    s1, s2 = O.selection_sums(la, dl, m1, m2, lnp, z_cat_max=zcat)
    xi_mc = s1 / N
    ne = O.neff(s1, s2, N)
    zD = min(O.z_of_dl(la, [D])[0], zcat)
    _, vmax = O.volume(la, [zcat])

    def f(z):
        dv, _ = O.volume(la, [z])
        return O.psi(la, [z])[0] * dv[0] / vmax[0] / (1 + z)
    xi_q, _ = integrate.quad(f, 0, zD, epsabs=0, epsrel=1e-10)
    assert ne > 2000
    assert abs(xi_mc - xi_q) < 4 * xi_q / math.sqrt(ne), (xi_mc, xi_q, ne)
    assert 4 / math.sqrt(ne) < 0.05                                 # the check resolves 5% (a dropped (1+z) is >20%)


# ------------------------------------------------------------------ P10: invariances
def _one_event(w, i):
    s = slice(w.sample_off[i], w.sample_off[i + 1])
    g = slice(w.grid_off[i], w.grid_off[i + 1])
    return w.dL[s], w.m1d[s], w.m2d[s], w.ln_prior[s], w.z_grid[g], w.p_gal[g]


def test_p10_weight_scaling_and_h0_rescaling():
    w = make_workload("tiny", n_samples=300)
    la = w.lam[0]
    dl, m1, m2, lp, zg, pg = _one_event(w, 0)
    a, h, _ = O.event_logI(la, dl, m1, m2, lp, zg, pg)
    b, h2, _ = O.event_logI(la, dl, m1, m2, lp - math.log(7.0), zg, pg)
    assert abs(b - a - math.log(7.0)) < 1e-12 and abs(h2 / h - 1) < 1e-13
    # (H0, dL) -> (a H0, dL/a): same z_j
    lb = la.copy()
    lb[0] *= 1.3
    z1, _, _ = O.sample_weights(la, dl, m1, m2, lp)
    z2, _, _ = O.sample_weights(lb, dl / 1.3, m1, m2, lp)
    assert np.allclose(z1, z2, rtol=0, atol=1e-12)


def test_p10_placements_converge_for_small_h():
    w = make_workload("tiny", n_samples=300)
    la = w.lam[0]
    dl, m1, m2, lp, zg, _ = _one_event(w, 1)
    zf = np.linspace(zg[0], zg[-1], 4001)
    pg = np.exp(-0.5 * ((zf - zf.mean()) / 0.05) ** 2)                 # smooth p_gal
    diffs = []
    for h in (4e-3, 1e-3):
        a, _, _ = O.event_logI(la, dl, m1, m2, lp, zf, pg, placement=O.PLACE_SAMPLES, bw_rule=O.BW_FIXED, fixed_bw=h)
        b, _, _ = O.event_logI(la, dl, m1, m2, lp, zf, pg, placement=O.PLACE_GRID, bw_rule=O.BW_FIXED, fixed_bw=h)
        diffs.append(abs(a - b))
    assert diffs[1] < diffs[0] / 8 and diffs[1] < 1e-4                  # O(h^2) convergence


def test_scott_bandwidth_reduces_to_textbook_for_equal_weights():
    rng = np.random.default_rng(5)
    z = rng.standard_normal(200) * 0.1 + 1.0
    h = O.scott_bw(z, np.full(200, 3.3))
    assert abs(h - np.std(z, ddof=1) * 200 ** -0.2) < 1e-14
    # duplicating a point == doubling its weight (Kish n_eff / reliability weights are not frequency
    # weights, so only check scale invariance and finiteness here)
    assert abs(O.scott_bw(z, np.full(200, 1e-20)) - h) < 1e-14
    assert math.isnan(O.scott_bw([0.3], [1.0])) and math.isnan(O.scott_bw(z, np.zeros(200)))


def test_scott_bandwidth_two_samples_closed_form_for_every_weight_ratio():
    # two samples d apart, weights (1, eps): sum w^2 = (1 + eps^2)/(1 + eps)^2 and sigma^2 = d^2/2 for EVERY eps > 0 (both sums
    # of the rule tend to 0 together: R21), so h = d/sqrt(2) n_eff^(-1/5); undefined only when the second weight IS zero
    d = 0.04
    for eps in (1.0, 0.1, 1e-3, 1e-4, 4e-5, 1e-12, 1e-30, 1e-300):
        s2 = (1 + eps ** 2) / (1 + eps) ** 2
        h = O.scott_bw([0.5, 0.5 + d], [1.0, eps])
        assert abs(h / (d / math.sqrt(2) * s2 ** 0.2) - 1) < 1e-12, eps
        assert abs(O.scott_bw([0.5 + d, 0.5], [eps, 1.0]) / h - 1) < 1e-12               # order of the samples
    for lr in (-800.0, -5000.0, -1e6):                                                      # ratios below the fp64 range
        assert abs(O.scott_bw_log([0.5, 0.5 + d], [3.0, 3.0 + lr]) / (d / math.sqrt(2)) - 1) < 1e-12
    assert math.isnan(O.scott_bw([0.5, 0.5 + d], [1.0, 0.0]))
    assert math.isnan(O.scott_bw_log([0.5, 0.5 + d], [-np.inf, -np.inf]))
    assert math.isnan(O.scott_bw([0.5, 0.5, 0.5], [1.0, 0.3, 0.2]))                        # zero variance


def test_scott_bandwidth_is_the_plain_rule_in_high_precision():
    # O7 as SURVEY writes it -- w^ = w/sum w, n_eff = 1/sum w^^2, var = sum w^(z - zbar)^2/(1 - sum w^^2) -- typed out with
    # 1000-digit arithmetic (mpmath: 1 - sum w^^2 is 10^-869 in the last case), against the oracle's cancellation-free rearrangement, on weights spanning 10^-40 .. 1,
    # on one dominant sample plus a sprinkle at 10^-25, and on weights that only exist as logs (e^-3000)
    import mpmath as mp
    mp.mp.dps = 1000
    rng = np.random.default_rng(11)

    def plain(z, lw):
        lw = [mp.mpf(float(x)) for x in lw]
        m = max(lw)
        w = [mp.e ** (x - m) for x in lw]
        sw = mp.fsum(w)
        wh = [x / sw for x in w]
        s2 = mp.fsum(x * x for x in wh)
        zb = mp.fsum(x * mp.mpf(float(t)) for x, t in zip(wh, z))
        var = mp.fsum(x * (mp.mpf(float(t)) - zb) ** 2 for x, t in zip(wh, z)) / (1 - s2)
        return float(mp.sqrt(var) * (1 / s2) ** mp.mpf(-0.2))
    z = 0.7 + 0.05 * rng.standard_normal(60)
    cases = [rng.uniform(-92.0, 0.0, 60),                                    # 40 decades
             np.concatenate([[0.0], rng.uniform(-60.0, -55.0, 59)]),         # one sample carries the event
             rng.uniform(-3000.0, -2990.0, 60),                              # all far below the fp64 range
             np.concatenate([[-700.0], rng.uniform(-2800.0, -2700.0, 59)])]  # both
    for lw in cases:
        assert abs(O.scott_bw_log(z, lw) / plain(z, lw) - 1) < 1e-12
    lw = cases[0]
    assert abs(O.scott_bw(z, np.exp(lw)) / plain(z, lw) - 1) < 1e-12       # the linear-weight entry is the same rule
    assert abs(O.scott_bw_log(z + 3.0, lw + 123.0) / O.scott_bw_log(z, lw) - 1) < 1e-12   # shift / scale invariance


def test_mass_function_in_log_space_matches_high_precision_deep_in_the_window():
    # ln S and ln p(m2|m1) where S itself leaves the fp64 range (m' < delta/709), against the definitions M1, M3 in
    # 40-digit arithmetic: S = 1/(1 + e^f), C(m1) = int m^beta S dm by mpmath's adaptive quadrature
    import mpmath as mp
    mp.mp.dps = 40
    la = lam()
    ml, dm, be = la[7], la[6], la[5]

    def S(m):
        mpr = mp.mpf(m) - mp.mpf(ml)
        return 1 / (1 + mp.e ** (mp.mpf(dm) / mpr + mp.mpf(dm) / (mpr - mp.mpf(dm))))
    for frac in (0.3, 0.02, 1.0 / 900.0, 1.0 / 3000.0):
        m = ml + frac * dm
        assert abs(O.ln_smoothing(la, [m])[0] / float(mp.log(S(m))) - 1) < 1e-12
        if frac > 1.0 / 700.0:
            assert abs(O.smoothing(la, [m])[0] / float(S(m)) - 1) < 1e-10            # the linear entry, where it exists
    for frac1, frac2 in ((0.5, 0.3), (0.05, 0.04), (1.0 / 500.0, 1.0 / 550.0), (1.0 / 2000.0, 1.0 / 2500.0), (3.0, 1.0 / 1500.0)):
        m1, m2 = ml + frac1 * dm, ml + frac2 * dm
        top = min(m1, ml + dm)
        pts = [mp.mpf(ml)] + [mp.mpf(top) - (mp.mpf(top) - mp.mpf(ml)) / 2 ** k for k in range(1, 30)] + [mp.mpf(top)]
        Cw = mp.quad(lambda x: x ** mp.mpf(be) * S(x), pts)
        Cm = Cw + ((mp.mpf(m1) ** (be + 1) - mp.mpf(top) ** (be + 1)) / (be + 1) if m1 > top else 0)
        ref = float(mp.mpf(be) * mp.log(m2) + mp.log(S(m2)) - mp.log(Cm))
        got = O.ln_p_m2_given_m1(la, [m1], [m2])[0]
        assert abs(got - ref) < 1e-9 * max(1.0, abs(ref)), (frac1, frac2, got, ref)
    # the joint density where the linear one underflows: ln p = ln p(m1) + ln p(m2|m1)
    m1, m2 = 30.0, ml + dm / 1500.0
    assert O.mass_pdf(la, [m1], [m2])[0] == 0.0 and O.ln_mass_pdf(la, [m1], [m2])[0] < -1400.0
    assert abs(O.ln_mass_pdf(la, [m1], [m2])[0] - (math.log(O.p_m1(la, [m1])[0]) + O.ln_p_m2_given_m1(la, [m1], [m2])[0])) < 1e-9


def test_p10_weight_scaling_at_the_edge_of_the_fp64_range():
    # P10 where linear weights die: ln_prior -> ln_prior + c multiplies every weight by e^-c; h must not move and log I must
    # shift by exactly -c, also when the weights sit near 1e-300 and when they lie far below the smallest double
    w = make_workload("tiny", n_samples=300)
    la = w.lam[0]
    dl, m1, m2, lp, zg, pg = _one_event(w, 2)
    a, h, fa = O.event_logI(la, dl, m1, m2, lp, zg, pg)
    assert fa == 0 and -60 < a < 0
    for c in (650.0, 1350.0, 5000.0):
        b, h2, fb = O.event_logI(la, dl, m1, m2, lp + c, zg, pg)
        assert fb == 0 and abs(b - (a - c)) < 1e-9 and abs(h2 / h - 1) < 1e-12, c
    # an event carried by secondaries deep in the smoothing window (S(m2) < 2^-1024 for all of them) is small, not empty
    z = O.z_of_dl(la, dl)
    m2deep = (la[7] + la[6] / np.linspace(900.0, 4000.0, dl.size)) * (1 + z)
    v, hd, fd = O.event_logI(la, dl, np.maximum(m1, m2deep), m2deep, lp, zg, pg)
    assert fd == 0 and np.isfinite(v) and v < -900 and hd > 0
    _, wlin, _ = O.sample_weights(la, dl, np.maximum(m1, m2deep), m2deep, lp)
    assert np.all(wlin == 0.0)                                                          # (what the linear weights see)


# ------------------------------------------------------------------ P11: brute force, independent route
def _brute_loglike(la, events, inj, n_inj_total, z_cat_max, fixed_h=None):
    """Independent re-computation with scipy (quad / brentq) on tiny inputs; placement N."""
    H0, Om, Xi0, n, al, be, dm, ml, mh, mu, sg, lg, ga, ka, zp = la
    E = lambda z: math.sqrt(Om * (1 + z) ** 3 + 1 - Om)
    dC = lambda z: integrate.quad(lambda x: C / H0 / E(x), 0, z, epsabs=0, epsrel=1e-13)[0]
    Xi = lambda z: Xi0 + (1 - Xi0) * (1 + z) ** (-n)
    dL = lambda z: Xi(z) * (1 + z) * dC(z)
    ddL = lambda z: (dL(z + 1e-5) - dL(z - 1e-5)) / 2e-5              # numerical derivative on purpose
    S = lambda m: 0.0 if m <= ml else (1.0 if m >= ml + dm else 1 / (1 + math.exp(min(700.0, dm / (m - ml) + dm / (m - ml - dm)))))
    PL = lambda m: (1 - al) * m ** (-al) / (mh ** (1 - al) - ml ** (1 - al)) if ml <= m <= mh else 0.0
    G = lambda m: math.exp(-0.5 * ((m - mu) / sg) ** 2) / (sg * math.sqrt(2 * math.pi))
    p1u = lambda m: ((1 - lg) * PL(m) + lg * G(m)) * S(m)
    Z1 = sum(integrate.quad(p1u, a, b, epsabs=0, epsrel=1e-12, limit=500)[0] for a, b in ((ml, ml + dm), (ml + dm, mu), (mu, mh), (mh, mh + 300)))
    Cn = lambda m1: sum(integrate.quad(lambda m: m ** be * S(m), a, b, epsabs=0, epsrel=1e-12, limit=500)[0]
                        for a, b in ((ml, min(m1, ml + dm)), (min(m1, ml + dm), m1)) if b > a)
    psi = lambda z: (1 + z) ** ga / (1 + ((1 + z) / (1 + zp)) ** (ga + ka))
    pm = lambda m1, m2: p1u(m1) / Z1 * m2 ** be * S(m2) / Cn(m1) if (ml <= m2 <= m1) else 0.0

    def weight(dl, m1d, m2d):
        z = optimize.brentq(lambda x: dL(x) - dl, 0, 10, xtol=1e-14, rtol=1e-15)
        return z, pm(m1d / (1 + z), m2d / (1 + z)) * psi(z) / ((1 + z) ** 3 * abs(ddL(z)))
    total = 0.0
    logI = []
    for (dls, m1s, m2s, lps, zg, pg) in events:
        zw = [weight(*t) for t in zip(dls, m1s, m2s)]
        z = np.array([t[0] for t in zw])
        w = np.array([t[1] for t in zw]) / np.exp(lps)
        if fixed_h is None:
            wh = w / w.sum()
            neff = 1 / np.sum(wh ** 2)
            zb = np.sum(wh * z)
            h = math.sqrt(np.sum(wh * (z - zb) ** 2) / (1 - np.sum(wh ** 2))) * neff ** -0.2
        else:
            h = fixed_h
        K = np.array([np.sum(w * np.exp(-0.5 * ((x - z) / h) ** 2)) for x in zg]) / (len(z) * h * math.sqrt(2 * math.pi))
        I = np.trapezoid(K * pg, zg)
        logI.append(math.log(I))
    total = sum(logI)
    Vmax = 4 * math.pi / 3 * dC(z_cat_max) ** 3
    ssum = 0.0
    for dl, m1d, m2d, lnp in zip(*inj):
        z, wgt = weight(dl, m1d, m2d)
        if z <= z_cat_max:
            ssum += wgt * (4 * math.pi * dC(z) ** 2 * C / H0 / E(z)) / Vmax / math.exp(lnp)
    xi = ssum / n_inj_total
    return total - len(events) * math.log(xi), np.array(logI), math.log(xi)


@pytest.mark.parametrize("fixed_h", [None, 0.01])
def test_p11_brute_force_two_events_three_samples(fixed_h):
    w = make_workload("tiny", n_events=2, n_samples=3, n_grid=40, n_inj_draw=60)
    la = w.lam[0].copy()
    la[2], la[3] = 1.4, 2.2                                        # exercise Xi(z)
    events = [_one_event(w, i) for i in range(2)]
    inj = (w.inj_dL, w.inj_m1d, w.inj_m2d, w.inj_ln_pdraw)
    ref_total, ref_logI, ref_logxi = _brute_loglike(la, events, inj, w.n_inj_total, w.z_cat_max, fixed_h)
    kw = {} if fixed_h is None else dict(bw_rule=O.BW_FIXED, fixed_bw=np.full(2, fixed_h))
    r = O.loglike_workload(w, lam=la, **kw)
    assert np.allclose(r["event_logI"][0], ref_logI, rtol=0, atol=2e-8)
    assert abs(r["logxi"][0] - ref_logxi) < 2e-8
    assert abs(r["loglike"][0] - ref_total) < 1e-7


def test_p11_trapezoid_against_simpson_on_refined_grid():
    # analytic p_gal, 20x finer grid + Simpson: the grid trapezoid is converged to ~1e-9 on Gaussians
    rng = np.random.default_rng(11)
    z, w = 0.5 + 0.02 * rng.standard_normal(25), rng.random(25)
    h = 0.008
    pg = lambda x: np.exp(-0.5 * ((x - 0.51) / 0.004) ** 2)
    zg = np.linspace(0.35, 0.65, 301)
    I = O.event_integral(lam(), zg, O.kde(z, w, h, zg), pg(zg))
    zf = np.linspace(0.35, 0.65, 6001)
    Is = integrate.simpson(O.kde(z, w, h, zf) * pg(zf), x=zf)
    assert abs(I / Is - 1) < 1e-9


# ------------------------------------------------------------------ Epanechnikov variant (NEXT-2; reading R19)
def test_epanechnikov_single_sample_shape_mass_and_variance():
    # one sample: K(z) = w (3/(4 hE)) (1 - u^2) on |u| <= 1, hE = sqrt(5) h: integrates to w, variance h^2 (R19), support 2 hE
    z0, w0, h = 0.5, 2.0, 0.02
    hE = math.sqrt(5.0) * h
    zg = np.array([z0, z0 + 0.5 * hE, z0 - 0.5 * hE, z0 + hE, z0 + 1.0001 * hE, z0 - 3 * hE])
    K = O.kde_epanechnikov(np.array([z0]), np.array([w0]), h, zg)
    assert np.allclose(K[:3], w0 * 0.75 / hE * np.array([1.0, 0.75, 0.75]), rtol=1e-14)
    assert abs(K[3]) < 1e-12 * K[0] and K[4] == 0.0 and K[5] == 0.0
    mass = integrate.quad(lambda x: O.kde_epanechnikov(np.array([z0]), np.array([w0]), h, np.array([x]))[0],
                          z0 - hE, z0 + hE, epsabs=1e-13)[0]
    var = integrate.quad(lambda x: (x - z0) ** 2 * O.kde_epanechnikov(np.array([z0]), np.array([w0]), h, np.array([x]))[0],
                         z0 - hE, z0 + hE, epsabs=1e-15)[0] / mass
    assert abs(mass - w0) < 1e-12 and abs(var / h ** 2 - 1) < 1e-10


def test_epanechnikov_flat_p_gal_gives_mean_weight_and_brute_force():
    # flat p_gal on a wide grid: I = (1/N_s) sum w_j up to the trapezoid error of a piecewise quadratic (O(dz^2/hE^2));
    # and the grid sum against the hand-expanded double sum
    rng = np.random.default_rng(5)
    z, w = 0.6 + 0.03 * rng.standard_normal(40), rng.random(40)
    h = 0.01
    hE = math.sqrt(5.0) * h
    zg = np.linspace(0.3, 0.9, 60001)
    I = O.event_integral(lam(), zg, O.kde_epanechnikov(z, w, h, zg), np.ones_like(zg))
    assert abs(I / np.mean(w) - 1) < 1e-6
    zg2 = np.linspace(0.45, 0.75, 31)
    K = O.kde_epanechnikov(z, w, h, zg2)
    brute = [sum(wj * 0.75 / hE * max(0.0, 1 - ((g - zj) / hE) ** 2) for zj, wj in zip(z, w)) / 40 for g in zg2]
    assert np.allclose(K, brute, rtol=1e-13, atol=1e-300)


def test_epanechnikov_end_to_end_uses_the_same_bandwidth_rule():
    # kernel=EPANECHNIKOV swaps O8 only: same z_j, w_j, h; log I from the Epanechnikov KDE on the event grid
    w = make_workload("tiny", n_events=2, n_samples=200, n_grid=150, n_inj_draw=200)
    la = w.lam[0]
    rg = O.loglike_workload(w, lam=la)
    re = O.loglike_workload(w, lam=la, kernel=O.KERNEL_EPANECHNIKOV)
    assert np.array_equal(rg["h"], re["h"]) and rg["logxi"][0] == re["logxi"][0]
    for i in range(2):
        s, g = slice(w.sample_off[i], w.sample_off[i + 1]), slice(w.grid_off[i], w.grid_off[i + 1])
        zj, wj, _ = O.sample_weights(la, w.dL[s], w.m1d[s], w.m2d[s], w.ln_prior[s])
        K = O.kde_epanechnikov(zj, wj, re["h"][0, i], w.z_grid[g])
        I = O.event_integral(la, w.z_grid[g], K, w.p_gal[g])
        assert abs(re["event_logI"][0, i] - math.log(I)) < 1e-13
    assert np.max(np.abs(re["event_logI"] - rg["event_logI"])) < 0.5     # same estimator up to the kernel shape
    O.loglike_workload(w, lam=la)                                        # (leaves the oracle on the Gaussian kernel)


# ------------------------------------------------------------------ many-1d kernel (NEXT-1; eq. 18, reading R20)
def test_many1d_singleton_groups_are_single1d():
    w = make_workload("tiny", n_events=3, n_samples=120, n_grid=90, n_inj_draw=300)
    r0 = O.loglike_workload(w)
    r1 = O.loglike_workload(w, group_off=np.arange(4), ln_factor=np.zeros(3))
    assert r1["loglike"][0] == r0["loglike"][0] and np.array_equal(r1["event_logI"], r0["event_logI"])


def test_many1d_pixel_sum_is_logsumexp_of_the_pixel_integrals():
    # I_g = sum_k F_k I_k (eq. 14's pixel sum with eq. 18's kernel): the total from the per-pixel log I of the same run
    w = split_into_pixels(make_workload("tiny", n_events=3, n_samples=400, n_grid=120, n_inj_draw=300), n_pix=4)
    r = O.loglike_workload(w)
    tot = 0.0
    for g in range(3):
        k = slice(w.group_off[g], w.group_off[g + 1])
        tot += math.log(np.sum(np.exp(w.ln_factor[k]) * np.exp(r["event_logI"][0, k])))
    assert abs(r["loglike"][0] - (tot - 3 * r["logxi"][0])) < 1e-10
    # a pixel without weight is not an empty event; an event whose pixels are all empty is
    lam2 = w.lam[0].copy()
    lam2[7], lam2[8] = 200.0, 300.0                                   # m_low above every source mass: all weights 0
    r2 = O.loglike_batch(lam2, w.sample_off, w.dL, w.m1d, w.m2d, w.ln_prior, w.grid_off, w.z_grid, w.p_gal,
                         group_off=w.group_off, ln_factor=w.ln_factor)            # (no injections: xi would be 0 too)
    assert r2["loglike"][0] == -np.inf and (r2["flags"][0] & O.F_EVENT_ZERO)


def test_many1d_with_shared_p_gal_and_fixed_bandwidth_equals_single1d():
    # pins the normalisation reading R20: per-pixel KDE divided by N_k, pixel factor N_k/N_s.  The KDE is linear in the
    # samples, so with one p_gal for all pixels and one fixed h the pixel sum IS the single-1d integral.
    w1 = make_workload("tiny", n_events=2, n_samples=500, n_grid=150, n_inj_draw=300)
    wp = split_into_pixels(w1, n_pix=5, same_p_gal=True)
    h = 0.01
    r1 = O.loglike_workload(w1, bw_rule=O.BW_FIXED, fixed_bw=np.full(2, h))
    rp = O.loglike_workload(wp, bw_rule=O.BW_FIXED, fixed_bw=np.full(10, h))
    assert abs(rp["loglike"][0] - r1["loglike"][0]) < 1e-10


def test_many1d_sparse_pixels_are_left_out_of_the_pixel_sum():
    # R24: a pixel with one sample (or one sample left with weight under this lambda) has no Scott bandwidth; it is left out
    # of the pixel sum -- the result is the one of the same event without that pixel -- and BW_DEGENERATE is raised
    w = split_into_pixels(make_workload("tiny", n_events=3, n_samples=400, n_grid=120, n_inj_draw=300), n_pix=4)
    ref = O.loglike_workload(w)
    s = slice(w.sample_off[0], w.sample_off[0] + 2)
    one = (w.dL[s][:1], w.m1d[s][:1], w.m2d[s][:1], w.ln_prior[s][:1], math.log(0.01))
    below = (w.dL[s], w.m1d[s], np.array([w.m2d[s][0], 1.0]), w.ln_prior[s], math.log(0.02))   # second sample below m_low
    w2 = append_pixels(w, 1, [one, below])
    assert w2.n_events == w.n_events + 2 and w2.group_off[-1] == w2.n_events
    r = O.loglike_workload(w2)
    assert abs(r["loglike"][0] - ref["loglike"][0]) < 1e-12
    assert r["flags"][0] == ref["flags"][0] | O.F_BW_DEGENERATE
    k = int(w.group_off[2])
    assert np.isnan(r["event_logI"][0, k]) and np.isnan(r["event_logI"][0, k + 1])
    # an event made of sparse pixels only has support but no estimate: NaN (as the single-1d kernel with one sample)
    w3 = append_pixels(w, 2, [one])
    w3.group_off = np.append(w3.group_off[:-1], [w3.n_events - 1, w3.n_events])      # ... as a fourth event of its own
    r3 = O.loglike_workload(w3)
    assert np.isnan(r3["loglike"][0]) and (r3["flags"][0] & O.F_BW_DEGENERATE)


# ------------------------------------------------------------------ p_cat from a galaxy list (NEXT-3; eq. 8, R22)
def test_pcat_against_scipy_quadrature_and_unit_mass():
    la = lam(H0=67.0, Om=0.31)
    rng = np.random.default_rng(3)
    zt = rng.uniform(0.2, 0.6, 7)
    st = 0.01 * (1 + zt) * rng.uniform(0.5, 2.0, 7)
    wg = rng.uniform(0.5, 2.0, 7)
    dv = lambda z: O.volume(la, np.array([z]))[0][0]                      # dV_c/dz, itself pinned by eq. 23
    gauss = lambda z, m, s: math.exp(-0.5 * ((z - m) / s) ** 2) / (s * math.sqrt(2 * math.pi))
    Z = [integrate.quad(lambda z: gauss(z, m, s) * dv(z), max(0.0, m - 12 * s), m + 12 * s, epsabs=0, epsrel=1e-13)[0]
         for m, s in zip(zt, st)]
    zg = np.linspace(0.1, 0.8, 29)
    ref = [sum(w * gauss(z, m, s) / zz for w, m, s, zz in zip(wg, zt, st, Z)) * dv(z) / wg.sum() for z in zg]
    assert np.allclose(O.pcat(la, zt, st, zg, wg), ref, rtol=1e-11, atol=1e-300)
    # each galaxy contributes unit mass: p_cat integrates to 1 over a grid that covers the catalogue; unit weights = w None
    zf = np.linspace(0.0, 1.2, 24001)
    assert abs(np.trapezoid(O.pcat(la, zt, st, zf, wg), zf) - 1) < 1e-9
    assert np.allclose(O.pcat(la, zt, st, zg), O.pcat(la, zt, st, zg, np.ones(7)), rtol=1e-15)


def test_pcat_narrow_galaxies_reduce_to_the_gaussian_mixture_and_h0_cancels():
    # sigma -> 0: dV_c/dz is constant across a galaxy, so it cancels against Z_g and p_cat -> sum_g w_g N / sum_g w_g
    la = lam(H0=70.0, Om=0.3)
    zt, st = np.array([0.5, 0.9]), np.array([1e-5, 2e-5])
    zg = np.array([0.5 - 1e-5, 0.5, 0.5 + 2e-5, 0.9, 0.9 + 3e-5])
    mix = 0.5 * sum(np.exp(-0.5 * ((zg - m) / s) ** 2) / (s * math.sqrt(2 * math.pi)) for m, s in zip(zt, st))
    assert np.allclose(O.pcat(la, zt, st, zg), mix, rtol=2e-4)
    z2 = np.linspace(0.3, 1.1, 9)
    assert np.allclose(O.pcat(la, zt, np.array([0.02, 0.03]), z2), O.pcat(lam(H0=35.0, Om=0.3), zt, np.array([0.02, 0.03]), z2), rtol=1e-13)


# ------------------------------------------------------------------ lambda-gradients (NEXT-4)
def test_gradient_zero_directions_h0_scaling_identity_and_step_independence():
    import dataclasses
    w = make_workload("tiny", n_events=3, n_samples=150, n_grid=60, n_inj_draw=400)
    la = w.lam[0].copy()
    la[2], la[3] = 1.3, 1.7                                            # Xi0 != 1 so that n matters
    f0, g = O.loglike_grad(w, la, rel_step=1e-2)
    assert abs(f0 - O.loglike_workload(w, lam=la)["loglike"][0]) < 1e-12
    # directions that provably do not matter: Xi0 = 1 -> n drops out of eq. 2; lambda_g = 0 -> mu_g, sigma_g drop out of eq. 20
    lb = la.copy(); lb[2] = 1.0
    assert abs(O.loglike_grad(w, lb)[1][3]) < 1e-9
    lc = la.copy(); lc[11] = 0.0
    gc = O.loglike_grad(w, lc)[1]
    assert abs(gc[9]) < 1e-9 and abs(gc[10]) < 1e-9
    # log L depends on H0 and on the distance scale of the data (events and injections, priors held fixed) through H0 x d_L only:
    # z_j = Z(H0 d_L,j) and every weight carries the same 1/|d d_L/dz| ~ H0, which cancels between sum_i log I_i and N log xi.
    # So H0 dlogL/dH0 = dlogL/dln(a) at a = 1 with all d_L -> a d_L -- the right side differentiates the DATA, not lambda
    def f_scaled(a):
        w2 = dataclasses.replace(w, dL=w.dL * a, inj_dL=w.inj_dL * a)
        return O.loglike_workload(w2, lam=la)["loglike"][0]
    e = 1e-2
    d1 = (f_scaled(1 + e) - f_scaled(1 - e)) / (2 * e)
    d2 = (f_scaled(1 + e / 2) - f_scaled(1 - e / 2)) / e
    assert abs(la[0] * g[0] - (4 * d2 - d1) / 3) < 1e-5 * max(1.0, abs(la[0] * g[0]))
    # the Richardson value does not hang on the step (O(h^4)): half the step, same gradient
    _, g2 = O.loglike_grad(w, la, rel_step=5e-3)
    scale = np.max(np.abs(g * la))
    assert np.max(np.abs((g - g2) * la)) < 1e-5 * scale
    # and agrees with a five-point stencil typed out here for one parameter (alpha)
    h = 1e-2 * la[4]
    fv = O.loglike_workload(w, lam=np.array([la + d * h * np.eye(15)[4] for d in (-2, -1, 1, 2)]))["loglike"]
    assert abs(g[4] - (fv[0] - 8 * fv[1] + 8 * fv[2] - fv[3]) / (12 * h)) < 1e-5 * scale / la[4]


# ------------------------------------------------------------------ completeness terms (NEXT-3; eq. 7, 9, 10; R25)
def test_pgal_completeness_limits_fR_against_scipy_and_unit_mass():
    la = lam(H0=67.0, Om=0.31)
    rng = np.random.default_rng(4)
    zt = rng.uniform(0.2, 1.0, 9)
    st = 0.01 * (1 + zt)
    zmax = 1.5
    zg = np.linspace(0.0, 1.6, 33)
    pcat = O.pcat(la, zt, st, zg)
    dv = lambda z: O.volume(la, np.array([z]))[0][0]
    vmax = O.volume(la, np.array([zmax]))[1][0]
    u = np.array([dv(z) / vmax if z <= zmax else 0.0 for z in zg])
    # P_compl = 1: complete catalogue -> p_gal = p_cat, f_R = 1;  P_compl = 0: nothing catalogued -> p_gal = u(z) of R6, f_R = 0
    p1, f1 = O.pgal(la, zmax, zt, st, [0.0, 2.0], [1.0, 1.0], zg)
    assert abs(f1 - 1) < 1e-12 and np.allclose(p1, pcat, rtol=1e-12, atol=1e-300)
    p0, f0 = O.pgal(la, zmax, zt, st, [0.0, 2.0], [0.0, 0.0], zg)
    assert f0 == 0 and np.allclose(p0, u, rtol=1e-12, atol=1e-300)
    # a completeness falling with z (piecewise linear, constant beyond its nodes): f_R = int P u dz by scipy, eq. 7 term by term
    zc, pc = np.array([0.1, 0.4, 0.9, 1.2]), np.array([0.95, 0.8, 0.3, 0.05])
    P = lambda z: float(np.interp(z, zc, pc))
    fr_ref = sum(integrate.quad(lambda z: P(z) * dv(z) / vmax, a, b, epsabs=0, epsrel=1e-12)[0]
                 for a, b in zip([0.0, 0.1, 0.4, 0.9, 1.2], [0.1, 0.4, 0.9, 1.2, zmax]))
    pg, fr = O.pgal(la, zmax, zt, st, zc, pc, zg)
    assert abs(fr - fr_ref) < 1e-11 and 0.1 < fr < 0.6
    assert np.allclose(pg, fr * pcat + (1 - np.array([P(z) for z in zg])) * u, rtol=1e-12, atol=1e-300)
    # unit mass: f_R + int (1 - P) u = 1 (all galaxies inside the grid)
    zf = np.linspace(0.0, zmax, 30001)
    pf, _ = O.pgal(la, zmax, zt, st, zc, pc, zf)
    assert abs(np.trapezoid(pf, zf) - 1) < 1e-8
    # only the shape of the cosmology matters (H0 cancels in u and in p_cat)
    p2, f2 = O.pgal(lam(H0=90.0, Om=0.31), zmax, zt, st, zc, pc, zg)
    assert abs(f2 - fr) < 1e-13 and np.allclose(p2, pg, rtol=1e-12, atol=1e-300)


# ------------------------------------------------------------------ sample binning (NEXT-2; reading R23)
def test_binning_conserves_moments_and_reduces_to_the_unbinned_kde():
    rng = np.random.default_rng(9)
    z, w = 0.5 + 0.05 * rng.standard_normal(300), rng.random(300)
    zb, wb = O.bin_samples(z, w, 37)
    assert len(zb) == 37 and abs(wb.sum() - w.sum()) < 1e-12 and abs((wb * zb).sum() - (w * z).sum()) < 1e-12
    assert np.all(np.diff(zb) > 0) and zb[0] >= z.min() and zb[-1] <= z.max()
    edges = np.linspace(z.min(), z.max(), 38)
    k = np.minimum(((z - z.min()) / ((z.max() - z.min()) / 37)).astype(int), 36)
    for b in (0, 5, 36):
        m = k == b
        assert abs(wb[b] - w[m].sum()) < 1e-13 and abs(zb[b] - (w[m] * z[m]).sum() / w[m].sum()) < 1e-13
        assert edges[b] - 1e-12 <= zb[b] <= edges[b + 1] + 1e-12
    z1, w1 = O.bin_samples(z, w, 1)
    assert abs(z1[0] - (w * z).sum() / w.sum()) < 1e-13 and abs(w1[0] - w.sum()) < 1e-12
    # one sample per bin at most (bins far narrower than the sample spacing): the binned estimator IS the unbinned one
    zs = np.sort(0.4 + 0.2 * rng.random(12))
    ws = rng.random(12)
    zb, wb = O.bin_samples(zs, ws, 200000)
    assert np.allclose(zb[wb > 0], zs, rtol=0, atol=1e-15) and np.allclose(wb[wb > 0], ws)


def test_binning_end_to_end_converges_quadratically_and_keeps_h_and_the_normalisation():
    w = make_workload("tiny", n_events=3, n_samples=1500, n_grid=200, n_inj_draw=300)
    r0 = O.loglike_workload(w)
    err = []
    for nb in (32, 64, 128, 256):
        r = O.loglike_workload(w, n_bins=nb)
        assert np.array_equal(r["h"], r0["h"]) and r["logxi"][0] == r0["logxi"][0]
        err.append(np.max(np.abs(r["event_logI"] - r0["event_logI"])))
    assert err[0] > err[1] > err[2] > err[3] and err[3] < 2e-3
    assert 2.5 < err[1] / err[2] < 6.0 and 2.5 < err[2] / err[3] < 6.0          # O(bin width^2)
    O.loglike_workload(w, lam=w.lam[:1])                                          # (leaves the oracle unbinned)


# ------------------------------------------------------------------ flags / degenerate cases
def test_flags_and_degenerate_cases():
    w = make_workload("tiny", n_events=2, n_samples=50, n_grid=60, n_inj_draw=200)
    bad = w.lam[0].copy()
    bad[1] = 1.5                                                    # Om outside (0, 1]
    r = O.loglike_workload(w, lam=np.stack([w.lam[0], bad]))
    assert r["flags"][1] & O.F_LAMBDA_DOMAIN and np.isnan(r["loglike"][1]) and np.isfinite(r["loglike"][0])
    # an event whose secondary masses are all below m_low has zero weight -> log I = -inf
    w.m2d[:50] = 1.0
    r = O.loglike_workload(w, lam=w.lam[0])
    assert r["flags"][0] & O.F_EVENT_ZERO and r["event_logI"][0, 0] == -np.inf and r["loglike"][0] == -np.inf
    # no injections: log xi := 0
    w2 = make_workload("tiny", n_events=2, n_samples=50, n_grid=60, n_inj_draw=200)
    r2 = O.loglike_batch(w2.lam[0], w2.sample_off, w2.dL, w2.m1d, w2.m2d, w2.ln_prior, w2.grid_off, w2.z_grid, w2.p_gal)
    assert r2["logxi"][0] == 0 and abs(r2["loglike"][0] - r2["event_logI"][0].sum()) < 1e-12


def test_log_likelihood_assembly_eq3():
    w = make_workload("tiny", n_events=3, n_samples=80, n_grid=60, n_inj_draw=400)
    r = O.loglike_workload(w)
    s1, s2 = O.selection_sums(w.lam[0], w.inj_dL, w.inj_m1d, w.inj_m2d, w.inj_ln_pdraw)
    assert abs(r["logxi"][0] - math.log(s1 / w.n_inj_total)) < 1e-13
    assert abs(r["loglike"][0] - (r["event_logI"][0].sum() - 3 * r["logxi"][0])) < 1e-11
    assert abs(r["neff"][0] - s1 * s1 / (s2 - s1 * s1 / w.n_inj_total)) < 1e-9
