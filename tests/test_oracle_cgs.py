"""Pins for oracle Part D: the paper's own table Q(H_th, B, n_e, T_e) in cgs units with H_th per cell
from eqs 13-14 and the cell's radius (L128-L136), and the Coulomb table Q_cc(n_e, T_i, T_e) (L147); readings C-22, C-23.
What a plausible mistake would break: the per-cell scale height (a wrong radius, Omega_K or enthalpy), the unit conversions
of the four table coordinates, the axis order, the conversion of the tabulated cgs rate to code units, the sign and the
per-kelvin form of the Coulomb table.  CPU only."""
import math

import numpy as np
import pytest

C, KB, ME, MP = 2.99792458e10, 1.380649e-16, 9.1093837015e-28, 1.67262192369e-24
SIGT, GMSUN = 6.6524587321e-25, 1.32712440018e26
MR = ME / MP
TH2K = ME * C * C / KB
AXC = [4, 5, 6, 7]                       # log H_th, log B, log n_e, log T_e
LO = [3.0, 0.0, 2.0, 2.0]                # the paper's ranges (L124)
HI = [12.0, 10.0, 25.0, 15.0]


def _conv(un):
    rg = GMSUN * un.mbh_msun / C ** 2
    return (rg / C) / (un.rho_scale_cgs * C ** 2)


def test_scale_height_per_cell_by_hand(oracle):
    """eqs 13-14 (L130-L136) at three radii, written out: H = c_s/Omega_K, c_s^2 = gamma P/(rho + u + P) with P = rho (Theta_e
    + Theta_i) m_e/m_p and u = P/(gamma - 1) (c = 1), Omega_K = 1/(r^{3/2} + a) in units of c/r_g."""
    un = oracle.Units()
    rg = GMSUN * 10.0 / C ** 2
    for r, the, thi in ((3.0, 2.0, 40.0), (10.0, 0.3, 3.0), (100.0, 0.03, 0.3)):
        p = (the + thi) * MR
        cs = math.sqrt((5.0 / 3.0) * p / (1.0 + 1.5 * p + p))
        assert oracle.hth_cm(un, the, thi, r) == pytest.approx(rg * cs * (r ** 1.5 + 0.9375), rel=1e-13)
    # H grows like r^{3/2} + a at fixed temperature and like the sound speed at fixed radius
    assert oracle.hth_cm(un, 1.0, 1.0, 40.0) / oracle.hth_cm(un, 1.0, 1.0, 10.0) == pytest.approx((40 ** 1.5 + 0.9375) / (10 ** 1.5 + 0.9375), rel=1e-13)
    assert oracle.hth_cm(un, 1e-4, 1e-4, 10.0) / oracle.hth_cm(un, 1e-6, 1e-6, 10.0) == pytest.approx(10.0, rel=1e-3)   # non-relativistic: c_s ~ sqrt(T)


def _linear_table(oracle, coef, n=(5, 4, 6, 5), coul3=None, **kw):
    g = np.meshgrid(*[np.linspace(LO[k], HI[k], n[k]) for k in range(4)], indexing="ij")
    T = (sum(c * a for c, a in zip(coef, g)) - 20.0).astype(np.float64)
    T32 = T.astype(np.float32)
    return oracle.Table(AXC, list(n), LO, HI, [T32], cgs=True, coul3=coul3, **kw), T32


def test_table_coordinates_and_units_with_a_linear_table(oracle):
    """Multilinear interpolation reproduces functions linear in the coordinates, so with log10 Q = a log H + b log B + c log n_e
    + d log T_e - 20 (unequal coefficients: a swapped axis fails) the looked-up rate must equal that expression of the cell's
    own H_th (eqs 13-14 with ITS radius), B = sqrt(4 pi b^2 rho_scale c^2) (L173), n_e = rho rho_scale/m_p (C-14) and
    T_e = Theta_e m_e c^2/k_B, converted to code units by t_g/(rho_scale c^2)."""
    un = oracle.Units()
    coef = (0.5, -0.25, 1.0, 0.125)          # exactly representable: node values carry only fp32 rounding (|y| < 64: 4e-6)
    tab, _ = _linear_table(oracle, coef)
    rng = np.random.default_rng(5)
    n = 400
    rho = 10 ** rng.uniform(-6, 0, n); bsq = 10 ** rng.uniform(-8, 0, n)
    the = 10 ** rng.uniform(-3, 1.5, n); thi = 10 ** rng.uniform(-3, 1.5, n); r = 10 ** rng.uniform(0.3, 2.5, n)
    o = oracle.step(tab, un, rho, bsq, the, thi, 1e-9, r=r, coulomb_mode=oracle.COULOMB_OFF, want_rates=True)
    rg = GMSUN * 10.0 / C ** 2
    p = (the + thi) * MR
    H = rg * np.sqrt((5.0 / 3.0) * p / (1.0 + 2.5 * p)) * (r ** 1.5 + 0.9375)
    B = np.sqrt(4.0 * np.pi * bsq * 3e-7 * C ** 2)
    ne = rho * 3e-7 / MP
    Te = the * TH2K
    y = coef[0] * np.log10(H) + coef[1] * np.log10(B) + coef[2] * np.log10(ne) + coef[3] * np.log10(Te) - 20.0
    assert (np.log10(H) > LO[0]).all() and (np.log10(H) < HI[0]).all() and o["diag"]["n_clamped"] == 0
    assert o["lam0"] == pytest.approx(10.0 ** y * _conv(un), rel=2e-5)       # fp32 node values: 4e-6 in y
    # without a radius array the scale height is taken at r_ref (C-6)
    o2 = oracle.step(tab, un, rho[:5], bsq[:5], the[:5], thi[:5], 1e-9, coulomb_mode=oracle.COULOMB_OFF, want_rates=True)
    H2 = H[:5] * (10 ** 1.5 + 0.9375) / (r[:5] ** 1.5 + 0.9375)
    y2 = y[:5] + coef[0] * (np.log10(H2) - np.log10(H[:5]))
    assert o2["lam0"] == pytest.approx(10.0 ** y2 * _conv(un), rel=2e-5)


def test_filler_is_part_a_at_every_node_and_step_is_node_exact(oracle):
    """orc_fill_total4_cgs stores the fp32 rounding of log10 of Part A's Q_total at every node; a cell placed exactly on a node
    (its radius chosen so that H_th hits the node) cools at Part A's rate for that node (node exactness, north_star pin)."""
    un = oracle.Units()
    n = [4, 3, 5, 6]
    lo, hi = [6.0, 2.0, 10.0, 7.0], [9.0, 6.0, 18.0, 11.5]
    T = oracle.fill_total4_cgs(n, lo, hi, nthreads=4)
    ax = [np.linspace(lo[k], hi[k], n[k]) for k in range(4)]
    for idx in ((0, 0, 0, 0), (3, 2, 4, 5), (1, 2, 3, 4), (2, 0, 1, 2), (3, 1, 0, 5)):
        H, B, ne, Te = (10.0 ** ax[k][idx[k]] for k in range(4))
        ref = oracle.cooling_cgs(H, B, ne, Te / TH2K)["total"]
        assert float(T[idx]) == np.float32(math.log10(ref))
    tab = oracle.Table(AXC, n, lo, hi, [T], cgs=True)
    rg = GMSUN * 10.0 / C ** 2
    cells = []
    for idx in ((1, 1, 2, 3), (2, 2, 3, 4), (3, 0, 1, 5), (1, 2, 4, 2)):
        H, B, ne, Te = (10.0 ** ax[k][idx[k]] for k in range(4))
        the = Te / TH2K
        thi = 2.5 * the
        p = (the + thi) * MR
        cs = math.sqrt((5.0 / 3.0) * p / (1.0 + 2.5 * p))
        r = (H / (rg * cs) - 0.9375) ** (2.0 / 3.0)
        assert r > 1.0
        cells.append((ne * MP / 3e-7, B ** 2 / (4.0 * math.pi * 3e-7 * C ** 2), the, thi, r, H, B, ne))
    rho, bsq, the, thi, r, H, B, ne = (np.array(x) for x in zip(*cells))
    o = oracle.step(tab, un, rho, bsq, the, thi, 1e-9, r=r, coulomb_mode=oracle.COULOMB_OFF, want_rates=True)
    ref = np.array([oracle.cooling_cgs(H[k], B[k], ne[k], the[k])["total"] for k in range(len(cells))]) * _conv(un)
    assert o["lam0"] == pytest.approx(ref, rel=1e-5)             # fp32 rounding of log10 Q (|y| < 40) and of the coordinates' round trip
    # and the analytic mode of the same table shape uses the cell's own H_th too
    oa = oracle.step(tab, un, rho, bsq, the, thi, 1e-9, r=r, coulomb_mode=oracle.COULOMB_OFF, want_rates=True, rate_mode=oracle.RATE_ANALYTIC)
    assert oa["lam0"] == pytest.approx(ref, rel=1e-9)


def test_coulomb_table3_is_eq15_per_kelvin(oracle):
    """L147: Q_cc(n_e, T_i, T_e).  The table stores log10 [Q_cc/(T_i - T_e)] (C-23); at its nodes the step's exchange equals
    eq 15 (oracle Part A.6, itself pinned against mpmath), its sign follows T_i - T_e, and it scales like n_e^2."""
    un = oracle.Units()
    n3, lo3, hi3 = [4, 5, 6], [10.0, 7.0, 7.0], [19.0, 11.0, 12.0]
    K3 = oracle.fill_coulomb3_cgs(un, n3, lo3, hi3)
    ax = [np.linspace(lo3[k], hi3[k], n3[k]) for k in range(3)]
    # by hand at one node: (3/2)(m_e/m_p) n_e^2 lnLambda c k_B sigma_T C(theta_e, theta_i)
    ne, ti, te = 10.0 ** ax[0][2], 10.0 ** ax[1][3], 10.0 ** ax[2][1]
    k = 1.5 * MR * ne * ne * 20.0 * C * KB * SIGT * oracle.coulomb_C(te / TH2K, ti / TH2K)
    assert float(K3[2, 3, 1]) == np.float32(math.log10(k))
    assert K3[3, 3, 1] - K3[2, 3, 1] == pytest.approx(2.0 * (ax[0][3] - ax[0][2]), abs=1e-5)        # n_e^2
    tab, _ = _linear_table(oracle, (0.0, 0.0, 0.0, 0.0), coul3=K3, c3lo=lo3, c3hi=hi3)
    cells = []
    for ia, ib, ic in ((1, 1, 4), (2, 4, 0), (3, 2, 2), (0, 0, 5)):
        ne, ti, te = 10.0 ** ax[0][ia], 10.0 ** ax[1][ib], 10.0 ** ax[2][ic]
        cells.append((ne * MP / 3e-7, te / TH2K, ti / TH2K))
    rho, the, thi = (np.array(x) for x in zip(*cells))
    o = oracle.step(tab, un, rho, np.full(4, 1e-4), the, thi, 1e-12, want_rates=True)              # coulomb_mode defaults to the 3-D table
    ref = np.array([oracle.coulomb_code(un, rho[k], the[k], thi[k]) for k in range(4)])
    assert o["qcc0"] == pytest.approx(ref, rel=1e-5)
    assert (np.sign(o["qcc0"]) == np.sign(thi - the)).all() and (o["qcc0"] != 0).sum() == 3        # cell 2 has T_i = T_e: exactly zero
    # zero exchange at T_i = T_e, bit for bit (north_star pin), through the per-kelvin form
    o = oracle.step(tab, un, rho, np.full(4, 1e-4), the, the.copy(), 1e3, nsub=3)
    assert np.array_equal(o["theta_e"], o["theta_i"])


def test_cgs_step_conserves_and_limits(oracle):
    """The update after the lookup is Part B's (pinned in test_oracle_step.py); here only that Part D feeds it the same way:
    energy leaves through radiation only, the 30 % limiter bites for a huge rate, clamping is counted."""
    un = oracle.Units()
    tab, _ = _linear_table(oracle, (0.0, 0.0, 2.0, 0.5))
    rng = np.random.default_rng(9)
    n = 500
    rho = 10 ** rng.uniform(-6, 0, n); bsq = 10 ** rng.uniform(-8, 0, n)
    the = 10 ** rng.uniform(-3, 1.5, n); thi = 10 ** rng.uniform(-3, 1.5, n); r = 10 ** rng.uniform(0.3, 2.5, n)
    vol = rng.uniform(0.5, 2.0, n)
    o = oracle.step(tab, un, rho, bsq, the, thi, 5.0, nsub=2, r=r, vol=vol, coulomb_mode=oracle.COULOMB_ANALYTIC)
    u0 = rho * (the + thi) * MR * 1.5
    u1 = rho * (o["theta_e"] + o["theta_i"]) * MR * 1.5
    assert (o["theta_e"] > 0).all() and (u1 <= u0 * (1 + 1e-14)).all()
    assert o["diag"]["lum_total"] == pytest.approx(float(((u0 - u1) * vol).sum() / 5.0), rel=1e-10)
    assert 0 < o["diag"]["n_limited"] < n
    far = oracle.step(tab, un, rho[:3] * 1e-20, bsq[:3], the[:3], thi[:3], 1e-3, r=r[:3], coulomb_mode=oracle.COULOMB_OFF)
    assert far["diag"]["n_clamped"] == 3                         # n_e below 1e2 cm^-3: clamped to the table edge
