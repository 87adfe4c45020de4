"""Pins for oracle Part A (analytic physics, eqs 1-15) against what the paper and
the mathematics fix: closed forms, limits, library special functions (scipy), golden
numbers from tests/golden/paper_pins.txt.  CPU only."""
import math
import os

import numpy as np
import pytest
from scipy import special as sp

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_pins.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 3:
            GOLD[line[0]] = (float(line[1]), float(line[2]))

# CODATA-2018 cgs, typed here independently of oracle/
C_, KB, ME, MP, QE, HPL = 2.99792458e10, 1.380649e-16, 9.1093837015e-28, 1.67262192369e-24, 4.80320471257e-10, 6.62607015e-27
SIGT, SIGSB = 6.6524587321e-25, 5.670374419e-5


def gold(name, value):
    ref, tol = GOLD[name]
    assert value == pytest.approx(ref, rel=tol), name


# ---------------------------------------------------------------- constants / units
def test_constants_and_units(oracle):
    un = oracle.Units()
    gold("mec2_over_kb", ME * C_ ** 2 / KB)
    gold("mp_over_me", MP / ME)
    gold("xM_coeff", 4 * math.pi * ME * C_ / (3 * QE))
    # n_e = rho rho_scale / m_p (C-14), B = sqrt(4 pi bsq rho_scale c^2) (L173)
    assert oracle.ne_cgs(un, 0.5) == pytest.approx(0.5 * 3e-7 / MP, rel=1e-14)
    assert oracle.bfield_gauss(un, 1e-2) == pytest.approx(math.sqrt(4 * math.pi * 1e-2 * 3e-7) * C_, rel=1e-14)
    # r_g, t_g through H_th = r_g c_s / Omega_K and the rate conversion
    th_e, th_i, r = 0.3, 2.0, 10.0
    mr = ME / MP
    p = (th_e + th_i) * mr
    cs = math.sqrt((5 / 3) * p / (1 + p / (2 / 3) + p))
    h = oracle.hth_cm(un, th_e, th_i, r)
    rg = h / (cs * (r ** 1.5 + 0.9375))
    gold("rg_10msun_cm", rg)
    # rate conversion t_g/(rho_scale c^2): node value minus log10 of cgs total
    q = oracle.cooling_cgs(un.hth_cm, oracle.bfield_gauss(un, 1e-3), oracle.ne_cgs(un, 1e-2), 0.5)["total"]
    conv = 10 ** oracle.node_total_log10(un, 1e-2, 0.5, 1e-3) / q
    gold("tg_10msun_s", conv * 3e-7 * C_ ** 2)


# ---------------------------------------------------------------- bremsstrahlung, eqs 1-2
def test_brems_scaling_and_limits(oracle):
    # exact n_e^2 scaling
    for th in (1e-4, 0.3, 1.0, 7.0):
        assert oracle.brems_cgs(3e10, th) / oracle.brems_cgs(1.0, th) == pytest.approx(9e20, rel=1e-14)
    # theta -> 0: the non-relativistic n^2 T^(1/2) law with the e-i coefficient of eq 2
    coeff = oracle.brems_cgs(1.0, 1e-12) / math.sqrt(1e-12)
    gold("brems_lowtheta_coeff", coeff)
    assert coeff == pytest.approx(1.48e-22 * 4 * math.sqrt(2 / math.pi ** 3), rel=1e-6)
    # logarithmic slope -> 1/2
    def slope(th):
        e = 1e-4
        return (math.log(oracle.brems_cgs(1, th * (1 + e))) - math.log(oracle.brems_cgs(1, th * (1 - e)))) / (math.log1p(e) - math.log1p(-e))
    assert slope(1e-6) == pytest.approx(0.5000017, abs=2e-6)
    assert slope(1e-3) == pytest.approx(0.50193, abs=2e-5)


def test_brems_branch_values_and_golden(oracle):
    # separate ee and ei at the branch point by using the two coefficient combinations
    lo = oracle.brems_cgs(1.0, 1.0 - 1e-15)
    hi = oracle.brems_cgs(1.0, 1.0)
    assert lo == pytest.approx(2.56e-22 * GOLD["fee_at_1_minus"][0] + 1.48e-22 * GOLD["fei_at_1_minus"][0], rel=1e-7)
    assert hi == pytest.approx(2.56e-22 * GOLD["fee_at_1_plus"][0] + 1.48e-22 * GOLD["fei_at_1_plus"][0], rel=1e-7)
    assert hi / lo - 1 == pytest.approx(0.0059, abs=3e-4)      # small jump at theta_e = 1
    gold("brems_theta_0p1", oracle.brems_cgs(1.0, 0.1))
    gold("brems_theta_2", oracle.brems_cgs(1.0, 2.0))
    gold("brems_theta_10", oracle.brems_cgs(1.0, 10.0))


# ---------------------------------------------------------------- Bessel functions
@pytest.mark.parametrize("x", [1e-5, 0.0316, 0.5, 1.0, 10.0, 59.3, 1e3, 1e6])
def test_bessel_scaled_vs_scipy(oracle, x):
    for nu in (0.0, 1.0, 2.0):
        assert oracle.bessel_k_scaled(nu, x) == pytest.approx(sp.kve(nu, x), rel=5e-14)
    assert oracle.bessel_k2_scaled(x) == pytest.approx(sp.kve(2, x), rel=5e-14)


def test_k2_tilde_and_threshold(oracle):
    for name, th in (("k2_ratio_theta_1", 1.0), ("k2_ratio_theta_10", 10.0), ("k2_ratio_theta_100", 100.0)):
        gold(name, oracle.k2_tilde(th) / (2 * th * th))
    th8 = KB * 1e8 / (ME * C_ ** 2)
    gold("theta_at_1e8K", th8)
    # literal threshold (C-12): <= 1e8 K uses 2 theta^2, just above uses K2
    assert oracle.k2_tilde(th8 * (1 - 1e-9)) == pytest.approx(2 * th8 ** 2, rel=1e-8)
    gold("k2_at_1e8K", oracle.k2_tilde(th8 * (1 + 1e-9)))
    assert oracle.k2_tilde(0.5) == pytest.approx(sp.kv(2, 2.0), rel=1e-13)


# ---------------------------------------------------------------- synchrotron, eqs 3-6
def test_iprime_formula_points(oracle):
    # eq 4 at x = 1: 4.0505*(1+0.4+0.5316)*exp(-1.8899)
    assert oracle.iprime(1.0) == pytest.approx(4.0505 * 1.9316 * math.exp(-1.8899), rel=1e-14)
    # x = 16^... choose x = 4096: x^(1/6)=4, x^(1/4)=8, x^(1/2)=64, x^(1/3)=16
    assert oracle.iprime(4096.0) == pytest.approx(4.0505 / 4 * (1 + 0.4 / 8 + 0.5316 / 64) * math.exp(-1.8899 * 16), rel=1e-13)


def _J_closed(xc):
    a = 1.8899
    tc = a * xc ** (1 / 3)
    G = lambda s: sp.gammaincc(s, tc) * sp.gamma(s)
    return 3 * 4.0505 * (G(5.5) / a ** 5.5 + 0.4 * G(4.75) / a ** 4.75 + 0.5316 * G(4.0) / a ** 4)


@pytest.mark.parametrize("xc", [1e-30, 1e-6, 0.03, 1.0, 10.0, 100.0, 1000.0, 3e4])
def test_synch_integral_closed_form(oracle, xc):
    assert oracle.synch_J(xc) == pytest.approx(_J_closed(xc), rel=1e-11)


def test_synch_integral_golden(oracle):
    gold("synch_J_0", oracle.synch_J(1e-40))
    for name, xc in (("synch_J_1", 1.0), ("synch_J_10", 10.0), ("synch_J_100", 100.0), ("synch_J_1000", 1000.0)):
        gold(name, oracle.synch_J(xc))


@pytest.mark.parametrize("H,B,ne,th", [(1.5e7, 1e6, 1e17, 1.0), (1e3, 10.0, 1e10, 0.05), (1e12, 1e8, 1e20, 30.0),
                                       (1.5e7, 3e3, 1e12, 0.0169), (1.5e7, 3e3, 1e12, 0.0168)])
def test_nu_c_solves_eq5(oracle, H, B, ne, th):
    q, nuc = oracle.synch_cgs(H, B, ne, th)
    te = th * ME * C_ ** 2 / KB
    xm = 4 * math.pi * ME * C_ * nuc / (3 * QE * B * th ** 2)
    eps = 4.43e-30 * 4 * math.pi * nuc * ne / oracle.k2_tilde(th) * oracle.iprime(xm)
    lhs = 2 * H * eps                                  # eq 5 without the common 2 pi R dR
    rhs = 2 * 2 * math.pi * nuc ** 2 * KB * te / C_ ** 2
    assert lhs == pytest.approx(rhs, rel=1e-12)
    # eq 6 assembled here from the pieces
    rj = 2 * math.pi * KB * te * nuc ** 3 / (3 * C_ ** 2 * H)
    s = 3 * QE * B * th ** 2 / (4 * math.pi * ME * C_)
    thin = 4.43e-30 * 4 * math.pi * ne * s * s * _J_closed(xm) / oracle.k2_tilde(th)
    assert q == pytest.approx(rj + thin, rel=1e-10)


def test_nu_c_monotone(oracle):
    base = oracle.synch_cgs(1e7, 1e5, 1e15, 0.8)[1]
    assert oracle.synch_cgs(1e8, 1e5, 1e15, 0.8)[1] > base
    assert oracle.synch_cgs(1e7, 1e5, 1e16, 0.8)[1] > base


def test_synch_optically_thin_limit(oracle):
    # H -> 0: nu_c -> 0, only the thin integral survives; theta >> 1 so K2 -> 2 theta^2
    ne, B, th = 1e12, 1e4, 300.0
    q, _ = oracle.synch_cgs(1e-30, B, ne, th)
    coeff = q / (ne * B * B * th * th)
    gold("synch_thin_coeff", coeff * oracle.k2_tilde(th) / (2 * th * th))
    gold("synch_textbook_coeff", coeff)
    assert 16 * SIGT * C_ / (8 * math.pi) == pytest.approx(GOLD["synch_textbook_coeff"][0], rel=1e-4)


# ---------------------------------------------------------------- Compton, eqs 7-9
def test_compton_limits(oracle):
    th, H = 0.5, 1e7
    nuc = 1e12
    x = HPL * nuc / (ME * C_ ** 2)
    # tau -> 0 => eta -> 1
    assert oracle.compton_eta(nuc, 1e-5, H, th) == pytest.approx(1.0, abs=1e-9)
    # P -> 1 => eta -> 3 theta / x (saturated)
    assert oracle.compton_eta(nuc, 1e25, H, th) == pytest.approx(3 * th / x, rel=1e-9)
    # hard photons (x >= 3 theta) are not enhanced (L99)
    assert oracle.compton_eta(3 * th * ME * C_ ** 2 / HPL * 1.001, 1e20, H, th) == 1.0
    # eta >= 1 everywhere on a scan, including PA > 1
    for ne in 10.0 ** np.arange(8, 26, 1.5):
        for t in (1e-3, 0.05, 0.5, 5.0, 30.0):
            assert oracle.compton_eta(1e11, ne, H, t) >= 1.0


def test_compton_series_sum(oracle):
    # C-1: eta = 1 + P(A-1) sum_{j<jm} (PA)^j with jm = ln(3 theta/x)/ln A; exact for integer jm
    th, H = 0.4, 1e7
    A = 1 + 4 * th + 16 * th * th
    for ne in (1e15, 1e17, 3e17, 1e19):
        tau = 2 * ne * SIGT * H
        P = 1 - math.exp(-tau)
        for jm in (1, 3, 7):
            x = 3 * th / A ** jm
            nuc = x * ME * C_ ** 2 / HPL
            series = 1 + P * (A - 1) * sum((P * A) ** j for j in range(jm))
            assert oracle.compton_eta(nuc, ne, H, th) == pytest.approx(series, rel=1e-10)
    # the printed exponent "1 - lnP/lnA" does NOT reproduce the series (documents the typo)
    assert oracle.compton_eta(nuc, ne, H, th, printed_exponent=True) != pytest.approx(series, rel=1e-3)


def test_compton_continuous_across_PA_1(oracle):
    th, H, nuc = 0.2, 1e7, 1e10
    A = 1 + 4 * th + 16 * th * th
    tau1 = -math.log(1 - 1 / A)                        # PA = 1
    ne1 = tau1 / (2 * SIGT * H)
    vals = [oracle.compton_eta(nuc, ne1 * (1 + d), H, th) for d in (-1e-6, -1e-10, 0.0, 1e-10, 1e-6)]
    assert max(vals) / min(vals) - 1 < 1e-4
    x = HPL * nuc / (ME * C_ ** 2)
    assert vals[2] == pytest.approx(1 + (1 / A) * (A - 1) * math.log(3 * th / x) / math.log(A), rel=1e-6)


# ---------------------------------------------------------------- bridge, eqs 11-12
def test_bridge_limits(oracle):
    H, th = 1e7, 0.1
    te = th * ME * C_ ** 2 / KB
    bb = 4 * SIGSB * te ** 4
    # optically thin: tiny Q_thin, tiny n_e  => Q_total -> Q_thin (L118)
    qthin = 1e-30 * bb / H
    assert oracle.bridge_cgs(H, 1.0, th, qthin) == pytest.approx(qthin, rel=1e-9)
    # optically thick in absorption: Q_total -> (8/3) sigma T^4 / (H tau)
    qthin = 1e12 * bb / H
    tau = 1e12 + 2 * 1.0 * SIGT * H
    assert oracle.bridge_cgs(H, 1.0, th, qthin) == pytest.approx((8 / 3) * SIGSB * te ** 4 / (H * tau), rel=1e-9)
    # scattering dominated: tau_sca >> 1 >> tau_abs
    ne = 1e22
    tau_sca = 2 * ne * SIGT * H
    tau_abs = 1e-3
    q = oracle.bridge_cgs(H, ne, th, tau_abs * bb / H)
    assert q == pytest.approx((bb / H) / (1.5 * (tau_abs + tau_sca) + math.sqrt(3) + 1 / tau_abs), rel=1e-13)


def test_total_assembly(oracle):
    H, B, ne, th = 1.5e7, 2e5, 3e16, 0.7
    d = oracle.cooling_cgs(H, B, ne, th)
    assert d["brems"] == pytest.approx(oracle.brems_cgs(ne, th), rel=1e-15)
    qs, nuc = oracle.synch_cgs(H, B, ne, th)
    assert d["synch"] == qs and d["nu_c"] == nuc
    assert d["eta"] == oracle.compton_eta(nuc, ne, H, th)
    assert d["thin"] == pytest.approx(d["brems"] + d["eta"] * d["synch"], rel=1e-15)      # eq 10
    assert d["total"] == pytest.approx(oracle.bridge_cgs(H, ne, th, d["thin"]), rel=1e-15)
    assert d["total"] < d["thin"]


# ---------------------------------------------------------------- scale height, eqs 13-14
def test_scale_height(oracle):
    un = oracle.Units()
    assert oracle.omega_k(4.0, 0.9375) == pytest.approx(1 / (8 + 0.9375), rel=1e-15)
    # cold limit: c_s^2 -> gamma P / rho
    mr = ME / MP
    h = oracle.hth_cm(un, 1e-6, 1e-6, 10.0)
    rg = GOLD["rg_10msun_cm"][0]
    assert h == pytest.approx(rg * math.sqrt(5 / 3 * 2e-6 * mr) * (10 ** 1.5 + 0.9375), rel=1e-5)
    # ultra-hot limit: c_s^2 -> gamma P/(u+P) = gamma - 1
    h = oracle.hth_cm(un, 1e9, 1e9, 10.0)
    assert h == pytest.approx(rg * math.sqrt(2 / 3) * (10 ** 1.5 + 0.9375), rel=1e-5)


# ---------------------------------------------------------------- Coulomb, eq 15
def _C_scipy(te, ti):
    xe, xi = 1 / te, 1 / ti
    xm = xe + xi
    s = te + ti
    return ((2 * s * s + 1) / s * sp.kve(1, xm) + 2 * sp.kve(0, xm)) / (sp.kve(2, xe) * sp.kve(2, xi))


def test_coulomb_coefficient(oracle):
    for name, (te, ti) in (("coulomb_C_1_1", (1, 1)), ("coulomb_C_0p1_10", (0.1, 10)), ("coulomb_C_1em3_1em3", (1e-3, 1e-3)),
                           ("coulomb_C_31p6_31p6", (31.6, 31.6)), ("coulomb_C_1em3_31p6", (1e-3, 31.6)), ("coulomb_C_0p01_1", (0.01, 1))):
        gold(name, oracle.coulomb_C(te, ti))
        assert oracle.coulomb_C(te, ti) == pytest.approx(_C_scipy(te, ti), rel=1e-12)
    # naive (unscaled) Bessel form where it does not underflow: exponentials cancel
    te, ti = 0.05, 0.2
    naive = ((2 * (te + ti) ** 2 + 1) / (te + ti) * sp.kv(1, 1 / te + 1 / ti) + 2 * sp.kv(0, 1 / te + 1 / ti)) / (sp.kv(2, 1 / te) * sp.kv(2, 1 / ti))
    assert oracle.coulomb_C(te, ti) == pytest.approx(naive, rel=1e-11)
    # symmetric in its arguments; small-theta asymptote sqrt(2/pi)(1/s+2)/sqrt(s)
    assert oracle.coulomb_C(0.3, 4.0) == pytest.approx(oracle.coulomb_C(4.0, 0.3), rel=1e-14)
    s = 2e-3
    assert oracle.coulomb_C(1e-3, 1e-3) == pytest.approx(math.sqrt(2 / math.pi) * (1 / s + 2) / math.sqrt(s), rel=5e-3)


def test_coulomb_rate(oracle):
    un = oracle.Units()
    gold("coulomb_pref_per_n2", oracle.coulomb_pref_cgs(un) / (3e-7 / MP) ** 2)
    assert oracle.coulomb_pref_cgs(un) / (3e-7 / MP) ** 2 == pytest.approx(1.5 * (ME / MP) * 20 * C_ * SIGT * ME * C_ ** 2, rel=1e-12)
    q = oracle.coulomb_code(un, 1e-2, 0.5, 5.0)
    assert q > 0                                       # ions hotter: electrons heated
    assert oracle.coulomb_code(un, 1e-2, 5.0, 0.5) < 0
    assert oracle.coulomb_code(un, 1e-2, 0.7, 0.7) == 0.0
    assert oracle.coulomb_code(un, 3e-2, 0.5, 5.0) / q == pytest.approx(9.0, rel=1e-13)    # rho^2
    # C-3: ion_theta_mass_ratio rescales theta_i inside the Bessel bracket only
    un2 = oracle.Units(ion_theta_mass_ratio=1836.15267344)
    q2 = oracle.coulomb_code(un2, 1e-2, 0.5, 5.0)
    assert q2 / q == pytest.approx(oracle.coulomb_C(0.5, 5.0 / 1836.15267344) / oracle.coulomb_C(0.5, 5.0), rel=1e-12)


# ---------------------------------------------------------------- table nodes
def test_node_functions(oracle):
    un = oracle.Units()
    rho, the, bsq, thi = 3e-3, 0.8, 2e-4, 6.0
    ne, B = oracle.ne_cgs(un, rho), oracle.bfield_gauss(un, bsq)
    conv = GOLD["tg_10msun_s"][0] / (3e-7 * C_ ** 2)
    d = oracle.cooling_cgs(un.hth_cm, B, ne, the)
    assert oracle.node_total_log10(un, rho, the, bsq) == pytest.approx(math.log10(d["total"] * conv), abs=1e-6)
    H = oracle.hth_cm(un, the, thi, un.r_ref_rg)
    d4 = oracle.cooling_cgs(H, B, ne, the)
    y = oracle.node_proc_log10(un, rho, the, bsq, thi)
    assert y[0] == pytest.approx(math.log10(d4["brems"] * conv), abs=1e-6)
    assert y[1] == pytest.approx(math.log10(d4["synch"] * conv), abs=1e-6)
    assert y[2] == pytest.approx(math.log10(d4["eta"]), abs=1e-12)
    # recombining the three processes gives back the total (eqs 10-12)
    q, fr = oracle.combine_code(un, rho, the, thi, 10 ** y[0], 10 ** y[1], 10 ** y[2])
    assert q == pytest.approx(d4["total"] * conv, rel=1e-5)
    assert sum(fr) == pytest.approx(1.0, rel=1e-13)
    # brems node is independent of bsq and Theta_i, exactly 2 log rho + g(Theta_e)
    y2 = oracle.node_proc_log10(un, rho * 10, the, bsq * 7, thi / 3)
    assert y2[0] - y[0] == pytest.approx(2.0, abs=1e-12)
