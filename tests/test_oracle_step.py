"""Pins for oracle Part B (interpolation + limited, sub-stepped update; PAPER.md L122-L124,
L181, L185, L197 and readings C-5..C-17): node-exactness, linear-exactness, a library
interpolator, brute force on tiny tables, conservation / positivity / limits of the update.
CPU only."""
import itertools
import math

import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

ME, MP = 9.1093837015e-28, 1.67262192369e-24
MR = ME / MP
AX3 = [0, 1, 2]            # (log rho, log Theta_e, log bsq)
AX4 = [0, 1, 2, 3]         # (..., log Theta_i)


def _rand_table(rng, n):
    return rng.uniform(-30.0, -2.0, size=n).astype(np.float32)


# ---------------------------------------------------------------- interpolation (B1, B2)
@pytest.mark.parametrize("n", [(5, 4, 6), (3, 3, 3, 3), (7, 2, 5, 4)])
def test_interp_exact_at_nodes_and_vs_scipy(oracle, n):
    rng = np.random.default_rng(1)
    nd = len(n)
    lo = [-6.0, -3.0, -8.0, -3.0][:nd]
    hi = [0.0, 1.5, 0.0, 1.5][:nd]
    T = _rand_table(rng, n)
    axes = [np.linspace(lo[k], hi[k], n[k]) for k in range(nd)]
    for idx in itertools.islice(itertools.product(*[range(m) for m in n]), 0, None, 7):
        y, cl = oracle.interp(n, lo, hi, T, [axes[k][idx[k]] for k in range(nd)])
        assert y == pytest.approx(float(T[idx]), abs=1e-12) and not cl
    rgi = RegularGridInterpolator(axes, T.astype(np.float64), method="linear")
    pts = np.stack([rng.uniform(lo[k], hi[k], 400) for k in range(nd)], axis=1)
    ref = rgi(pts)
    for p, r in zip(pts, ref):
        y, cl = oracle.interp(n, lo, hi, T, list(p))
        assert y == pytest.approx(r, abs=1e-11) and not cl
        corners = T  # interpolant bounded by table extrema (weights in [0,1], sum 1)
        assert corners.min() - 1e-9 <= y <= corners.max() + 1e-9


def test_interp_linear_functions_exact(oracle):
    n, lo, hi = (9, 7, 5, 6), [-6.0, -3.0, -8.0, -3.0], [0.0, 1.5, 0.0, 1.5]
    axes = np.meshgrid(*[np.linspace(lo[k], hi[k], n[k]) for k in range(4)], indexing="ij")
    coef = [2.0, 0.5, -0.25, 1.0]
    # choose coefficients/nodes so that node values are exactly representable in fp32
    T = (4.0 + sum(c * np.round(a * 8) / 8 for c, a in zip(coef, axes))).astype(np.float32)
    rng = np.random.default_rng(2)
    lin = lambda x: 4.0 + sum(c * xi for c, xi in zip(coef, x))
    # node coordinates were rounded to multiples of 1/8 only if they already are: use exact grid
    n2, lo2, hi2 = (7, 5, 9, 4), [-6.0, -3.0, -8.0, -1.5], [0.0, 1.0, 0.0, 1.5]
    axes2 = np.meshgrid(*[np.linspace(lo2[k], hi2[k], n2[k]) for k in range(4)], indexing="ij")
    T2 = (4.0 + sum(c * a for c, a in zip(coef, axes2))).astype(np.float32)   # steps of 1, 1, 1, 1: exact
    for _ in range(300):
        x = [rng.uniform(lo2[k], hi2[k]) for k in range(4)]
        y, _cl = oracle.interp(n2, lo2, hi2, T2, x)
        assert y == pytest.approx(lin(x), abs=1e-12)


def test_interp_clamps_to_edge(oracle):
    rng = np.random.default_rng(3)
    n, lo, hi = (4, 5, 3), [-6.0, -3.0, -8.0], [0.0, 1.5, 0.0]
    T = _rand_table(rng, n)
    inside, _ = oracle.interp(n, lo, hi, T, [-6.0, 0.3, -8.0])
    out, cl = oracle.interp(n, lo, hi, T, [-9.5, 0.3, -20.0])
    assert cl and out == inside
    inside, _ = oracle.interp(n, lo, hi, T, [0.0, 1.5, -2.0])
    out, cl = oracle.interp(n, lo, hi, T, [0.7, 1e3, -2.0])
    assert cl and out == inside
    out, cl = oracle.interp(n, lo, hi, T, [-math.inf, 0.3, -8.0])          # non-positive primitive
    assert cl and out == oracle.interp(n, lo, hi, T, [-6.0, 0.3, -8.0])[0]
    assert math.isnan(oracle.interp(n, lo, hi, T, [math.nan, 0.3, -8.0])[0])


def test_interp_brute_force_formula(oracle):
    """y = sum_corners prod(w) T written out directly on a 3^3 and a 3^4 table."""
    rng = np.random.default_rng(4)
    for n in ((3, 3, 3), (3, 3, 3, 3)):
        nd = len(n)
        lo, hi = [0.0] * nd, [2.0] * nd       # node spacing 1: t = x
        T = _rand_table(rng, n)
        for _ in range(200):
            x = rng.uniform(0, 2, nd)
            i = np.minimum(np.floor(x).astype(int), 1)
            w = x - i
            ref = 0.0
            for c in itertools.product((0, 1), repeat=nd):
                pw = np.prod([w[k] if c[k] else 1 - w[k] for k in range(nd)])
                ref += pw * float(T[tuple(i + np.array(c))])
            assert oracle.interp(n, lo, hi, T, list(x))[0] == pytest.approx(ref, abs=1e-12)


# ---------------------------------------------------------------- the update (B3-B6)
def _const_table(oracle, log_lambda, coul_logC=None, ndim=3):
    n = [3] * ndim
    lo = [-6.0, -3.0, -8.0, -3.0][:ndim]
    hi = [0.0, 1.5, 0.0, 1.5][:ndim]
    data = [np.full(n, log_lambda, dtype=np.float32)]
    if coul_logC is None:
        return oracle.Table(AX4[:ndim], n, lo, hi, data)
    return oracle.Table(AX4[:ndim], n, lo, hi, data, coul=np.full((3, 3), coul_logC, np.float32),
                        clo=[-3.0, -3.0], chi=[1.5, 1.5])


def _cells(n, seed=5):
    rng = np.random.default_rng(seed)
    return (10 ** rng.uniform(-6, 0, n), 10 ** rng.uniform(-8, 0, n),
            10 ** rng.uniform(-3, 1.5, n), 10 ** rng.uniform(-3, 1.5, n))


def _u(rho, th, gam=5 / 3):
    return rho * th * MR / (gam - 1)


def test_update_conservation_positivity_diag(oracle):
    un = oracle.Units()
    rho, bsq, the, thi = _cells(2000)
    vol = np.random.default_rng(6).uniform(0.5, 2.0, rho.size)
    tab = _const_table(oracle, -9.0, coul_logC=0.0)
    for nsub in (1, 4):
        dt = 5.0
        o = oracle.step(tab, un, rho, bsq, the, thi, dt, nsub=nsub, vol=vol, want_rates=True)
        ue, ui = _u(rho, the), _u(rho, thi)
        ue2, ui2 = _u(rho, o["theta_e"]), _u(rho, o["theta_i"])
        assert (ue2 > 0).all() and (ui2 > 0).all()
        # total energy changes only by the radiated part; the diagnostic is its volume integral
        lost = (ue + ui) - (ue2 + ui2)
        assert (lost >= -1e-14 * (ue + ui)).all()
        assert o["diag"]["lum_total"] == pytest.approx(float((lost * vol).sum() / dt), rel=1e-10)
        assert 0 < o["diag"]["n_limited"] < rho.size
        assert o["diag"]["n_floored"] == 0
        if nsub == 1:
            assert o["diag"]["n_clamped"] == 0      # inputs are inside the table range
        assert o["lam0"] == pytest.approx(1e-9, rel=1e-12)


def test_update_strong_cooling_limit(oracle):
    """Lambda -> inf, Coulomb off: u_e' = 0.7^nsub u_e (30 % limiter, L185), ions untouched."""
    un = oracle.Units()
    rho, bsq, the, thi = _cells(300)
    tab = _const_table(oracle, 30.0)
    for nsub in (1, 2, 4):
        o = oracle.step(tab, un, rho, bsq, the, thi, 1e-3, nsub=nsub, coulomb_mode=oracle.COULOMB_OFF)
        assert o["theta_e"] == pytest.approx(the * 0.7 ** nsub, rel=1e-13)
        assert o["theta_i"] == pytest.approx(thi, rel=1e-15)
        assert o["diag"]["n_limited"] == rho.size
    o = oracle.step(tab, un, rho, bsq, the, thi, 1e-3, nsub=1, f_limit=0.1, coulomb_mode=oracle.COULOMB_OFF)
    assert o["theta_e"] == pytest.approx(the * 0.9, rel=1e-13)


def test_update_constant_rate_independent_of_nsub(oracle):
    un = oracle.Units()
    rho, bsq, the, thi = _cells(300)
    tab = _const_table(oracle, -16.0)
    a = oracle.step(tab, un, rho, bsq, the, thi, 1e-3, nsub=1, coulomb_mode=oracle.COULOMB_OFF)
    b = oracle.step(tab, un, rho, bsq, the, thi, 1e-3, nsub=4, coulomb_mode=oracle.COULOMB_OFF)
    assert a["diag"]["n_limited"] == 0
    assert a["theta_e"] == pytest.approx(b["theta_e"], rel=1e-13)
    # du_e = -Lambda dt exactly
    assert _u(rho, the) - _u(rho, a["theta_e"]) == pytest.approx(1e-16 * 1e-3, rel=1e-6)


def test_update_small_dt_derivative(oracle):
    """dt -> 0: (u' - u)/dt -> -Lambda + Q_cc for electrons, -Q_cc for ions."""
    un = oracle.Units()
    rho, bsq, the, thi = _cells(200)
    tab = _const_table(oracle, -14.0, coul_logC=-0.3)
    dt = 1e-6
    o = oracle.step(tab, un, rho, bsq, the, thi, dt, want_rates=True)
    pref = oracle.coulomb_pref_cgs(un) * 4.925491e-5 / (3e-7 * 2.99792458e10 ** 2)
    qcc = pref * rho ** 2 * (thi - the) * 10 ** -0.3
    assert o["qcc0"] == pytest.approx(qcc, rel=2e-6)
    assert o["lam0"] == pytest.approx(1e-14, rel=1e-12)
    ue, ui = _u(rho, the), _u(rho, thi)
    due = (_u(rho, o["theta_e"]) - ue) / dt
    dui = (_u(rho, o["theta_i"]) - ui) / dt
    ok = (np.abs(qcc) * dt < 1e-3 * np.minimum(ue, ui)) & (1e-14 * dt < 1e-3 * ue)   # limiter idle
    assert ok.sum() > 50
    # an unlimited explicit step is exactly linear in dt: only rounding of u remains
    assert (np.abs(due - (-1e-14 + qcc)) <= 1e-6 * (1e-14 + np.abs(qcc)) + 8e-16 * ue / dt)[ok].all()
    assert (np.abs(dui + qcc) <= 1e-6 * np.abs(qcc) + 8e-16 * ui / dt)[ok].all()
    # and the rates are visible above the rounding noise for a good share of the cells
    assert ((1e-14 + np.abs(qcc)) > 1e3 * 8e-16 * ue / dt)[ok].sum() > 20


def test_coulomb_alone_no_crossing_and_zero_at_equality(oracle):
    un = oracle.Units()
    rho, bsq, the, thi = _cells(500)
    tab = _const_table(oracle, -300.0, coul_logC=6.0)          # no radiation, violent exchange
    o = oracle.step(tab, un, rho, bsq, the, thi, 1e3, nsub=8)
    s0 = np.sign(thi - the)
    d1 = o["theta_i"] - o["theta_e"]
    d1[np.abs(d1) < 1e-14 * o["theta_i"]] = 0.0               # equalised up to rounding
    s1 = np.sign(d1)
    assert ((s1 == s0) | (s1 == 0)).all()                      # temperatures never cross
    assert (np.abs(o["theta_i"] - o["theta_e"]) <= np.abs(thi - the) * (1 + 1e-12)).all()
    # total energy conserved by the exchange
    assert _u(rho, o["theta_e"]) + _u(rho, o["theta_i"]) == pytest.approx(_u(rho, the) + _u(rho, thi), rel=1e-12)
    # after many strong sub-steps a good fraction has equalised exactly
    assert (np.abs(o["theta_i"] / o["theta_e"] - 1) < 1e-12).mean() > 0.3
    # exact zero exchange at T_e = T_i (north_star pin)
    o = oracle.step(tab, un, rho, bsq, the, the.copy(), 1e3, nsub=3)
    assert (o["theta_e"] == o["theta_i"]).all()
    assert o["theta_e"] == pytest.approx(the, rel=1e-15)
    # analytic Coulomb too
    tab2 = _const_table(oracle, -300.0)
    o = oracle.step(tab2, un, rho[:20], bsq[:20], the[:20], the[:20].copy(), 1e3, coulomb_mode=oracle.COULOMB_ANALYTIC)
    assert (o["theta_e"] == o["theta_i"]).all() and o["theta_e"] == pytest.approx(the[:20], rel=1e-15)


def test_equalising_transfer_unequal_gammas(oracle):
    un = oracle.Units(gamma_e=4.0 / 3.0, gamma_i=5.0 / 3.0)
    rho, bsq, the, thi = _cells(200)
    tab = _const_table(oracle, -300.0, coul_logC=12.0)
    o = oracle.step(tab, un, rho, bsq, the, thi, 1e6, nsub=40, f_limit=0.45)
    assert o["theta_e"] == pytest.approx(o["theta_i"], rel=1e-9)   # converge to common Theta
    etot0 = _u(rho, the, 4 / 3) + _u(rho, thi, 5 / 3)
    etot1 = _u(rho, o["theta_e"], 4 / 3) + _u(rho, o["theta_i"], 5 / 3)
    assert etot1 == pytest.approx(etot0, rel=1e-12)


def test_floor_switches_cooling_off(oracle):
    """eq 19 (L195): T_gas = p/rho below (pi/2)(h_floor Omega_K r)^2 => no cooling."""
    un = oracle.Units()
    n = 400
    rho, bsq, _, _ = _cells(n)
    r = np.full(n, 20.0)
    tfloor = 0.5 * math.pi * (0.1 * 20.0 / (20.0 ** 1.5 + 0.9375)) ** 2
    th_tot = tfloor / MR * np.linspace(0.5, 1.5, n)               # straddles the floor
    the, thi = 0.25 * th_tot, 0.75 * th_tot
    tab = _const_table(oracle, -6.0)
    o = oracle.step(tab, un, rho, bsq, the, thi, 1e-2, h_floor=0.1, r=r, coulomb_mode=oracle.COULOMB_OFF)
    below = (the + thi) * MR < tfloor
    assert below.sum() > 100 and (~below).sum() > 100
    assert o["theta_e"][below] == pytest.approx(the[below], rel=1e-15)
    assert (o["theta_e"][~below] < the[~below]).all()
    assert o["diag"]["n_floored"] == int(below.sum())
    o2 = oracle.step(tab, un, rho, bsq, the, thi, 1e-2, h_floor=0.0, r=r, coulomb_mode=oracle.COULOMB_OFF)
    assert (o2["theta_e"] < the).all()


def test_passthrough_and_nan(oracle):
    un = oracle.Units()
    tab = _const_table(oracle, -6.0, coul_logC=0.0)
    rho = np.array([0.0, -1.0, 1e-3, np.nan, 1e-3])
    bsq = np.array([1e-4, 1e-4, 0.0, 1e-4, 1e-4])
    the = np.array([0.5, 0.5, 0.5, 0.5, np.nan])
    thi = np.array([2.0, 2.0, 2.0, 2.0, 2.0])
    o = oracle.step(tab, un, rho, bsq, the, thi, 1e-3)
    assert o["theta_e"][0] == 0.5 and o["theta_i"][1] == 2.0           # rho <= 0: unchanged
    assert np.isfinite(o["theta_e"][2]) and o["theta_e"][2] != 0.5     # bsq = 0 clamps to lower edge
    assert np.isnan(o["theta_e"][3]) and np.isnan(o["theta_e"][4])     # NaN in, NaN out, that cell only
    assert o["diag"]["n_clamped"] == 1


def test_table_step_reproduces_analytic_at_nodes(oracle):
    """Exact reproduction at table nodes (north_star pin) + brute force on a tiny grid:
    cells that sit exactly on nodes of an oracle-filled table give the analytic step."""
    un = oracle.Units()
    n, lo, hi = [4, 5, 4], [-5.0, -2.0, -6.0], [-2.0, 1.0, -3.0]      # node spacing 1, 0.75, 1 dex
    T = oracle.fill_total3(un, n, lo, hi, nthreads=4)
    tab = oracle.Table(AX3, n, lo, hi, [T])
    g = np.meshgrid(*[np.linspace(lo[k], hi[k], n[k]) for k in range(3)], indexing="ij")
    rho, the, bsq = (10 ** a.ravel() for a in g)
    thi = 3.0 * the
    a = oracle.step(tab, un, rho, bsq, the, thi, 1e-3, coulomb_mode=oracle.COULOMB_OFF, want_rates=True)
    b = oracle.step(tab, un, rho, bsq, the, thi, 1e-3, coulomb_mode=oracle.COULOMB_OFF, want_rates=True,
                    rate_mode=oracle.RATE_ANALYTIC)
    assert a["lam0"] == pytest.approx(b["lam0"], rel=3e-6)        # fp32 rounding of log10 Lambda (|y|<~40)
    assert a["theta_e"] == pytest.approx(b["theta_e"], rel=1e-6)
    # and the stored node is the fp32 rounding of the analytic value
    k = 37
    idx = np.unravel_index(k, n)
    assert float(T[idx]) == np.float32(oracle.node_total_log10(un, rho[k], the[k], bsq[k]))


def test_process_tables_and_luminosity_split(oracle):
    """nproc = 3 (config 5): per-process tables recombined by eqs 10-12 with the cell's H;
    luminosity shares add up to the total."""
    un = oracle.Units()
    n, lo, hi = [3, 4, 3, 3], [-4.0, -1.5, -5.0, -1.0], [-2.0, 1.5, -3.0, 1.0]
    g = np.meshgrid(*[np.linspace(lo[k], hi[k], n[k]) for k in range(4)], indexing="ij")
    nodes = np.stack([10 ** a.ravel() for a in g], axis=1)
    vals = np.array([oracle.node_proc_log10(un, *row) for row in nodes], dtype=np.float32)
    data = [vals[:, p].reshape(n) for p in range(3)]
    tab = oracle.Table(AX4, n, lo, hi, data)
    rho, the, bsq, thi = nodes.T
    a = oracle.step(tab, un, rho, bsq, the, thi, 1e-2, coulomb_mode=oracle.COULOMB_OFF, want_rates=True)
    b = oracle.step(tab, un, rho, bsq, the, thi, 1e-2, coulomb_mode=oracle.COULOMB_OFF, want_rates=True,
                    rate_mode=oracle.RATE_ANALYTIC)
    assert a["lam0"] == pytest.approx(b["lam0"], rel=1e-5)
    d = a["diag"]
    assert d["lum_brems"] + d["lum_synch"] + d["lum_compton"] == pytest.approx(d["lum_total"], rel=1e-12)
    assert d["lum_brems"] > 0 and d["lum_synch"] > 0 and d["lum_compton"] >= 0


def test_cell_luminosity_terms_and_shell_sums(oracle):
    """Per-cell terms of eq 22 (L222) and their shell sums (eq 25): each cell's term equals the energy it lost
    (energy leaves only through radiation), the terms add up to the whole-field diagnostic, the per-process terms add up
    to the total, and shell sums are partial sums."""
    un = oracle.Units()
    rng = np.random.default_rng(31)
    n = [4, 5, 3, 4]
    data = [rng.uniform(-12.0, -7.0, size=n).astype(np.float32), rng.uniform(-12.0, -7.0, size=n).astype(np.float32),
            rng.uniform(0.0, 1.0, size=n).astype(np.float32)]
    tab = oracle.Table(AX4, n, [-6.0, -3.0, -8.0, -3.0], [0.0, 1.5, 0.0, 1.5], data,
                       coul=np.zeros((3, 3), np.float32), clo=[-3.0, -3.0], chi=[1.5, 1.5])
    rho, bsq, the, thi = _cells(1200, seed=32)
    vol = rng.uniform(0.5, 2.0, rho.size)
    dt = 7.0
    for fn, kw in ((oracle.step, dict(nsub=3)), (oracle.step_implicit, dict(nsub=2))):
        o = fn(tab, un, rho, bsq, the, thi, dt, vol=vol, want_cell_lum=True, **kw)
        cl = o["cell_lum"]
        lost = (_u(rho, the) + _u(rho, thi)) - (_u(rho, o["theta_e"]) + _u(rho, o["theta_i"]))
        assert cl[:, 0] == pytest.approx(lost * vol / dt, rel=1e-9, abs=1e-14 * float((lost * vol / dt).max()))
        assert cl[:, 1:].sum(axis=1) == pytest.approx(cl[:, 0], rel=1e-12)
        assert (cl >= 0).all() and (cl[:, 0] > 0).sum() > 1000
        d = o["diag"]
        assert cl.sum(axis=0) == pytest.approx([d["lum_total"], d["lum_brems"], d["lum_synch"], d["lum_compton"]], rel=1e-12)
        sh = oracle.shell_sums(cl, 256)
        assert sh.shape == (5, 4)
        assert sh[2] == pytest.approx(cl[512:768].sum(axis=0), rel=1e-13)
        assert sh[4] == pytest.approx(cl[1024:].sum(axis=0), rel=1e-13)          # ragged last shell


# ---------------------------------------------------------------- per-process luminosity split (reading C-21)
# DESIGN.md C-21: the energy a cell radiates is attributed to bremsstrahlung, synchrotron and the Compton-added part in
# proportion to their shares of Q_thin = Q_brem + eta Q_syn (eq 10): Q_brem, Q_syn, (eta - 1) Q_syn;
# the optically-thick bridge of eqs 11-12 (L108-L118) and the limiter (L185) scale all three alike.
def _proc_table(oracle, log_br, log_sy, log_eta, with_coul=False):
    n = [3, 3, 3, 3]
    lo, hi = [-6.0, -3.0, -8.0, -3.0], [0.0, 1.5, 0.0, 1.5]
    data = [np.full(n, v, dtype=np.float32) for v in (log_br, log_sy, log_eta)]
    if with_coul:
        return oracle.Table(AX4, n, lo, hi, data, coul=np.zeros((3, 3), np.float32), clo=[-3.0, -3.0], chi=[1.5, 1.5])
    return oracle.Table(AX4, n, lo, hi, data)


def _both_schemes(oracle, tab, un, rho, bsq, the, thi, dt, vol, nsub):
    yield "explicit", oracle.step(tab, un, rho, bsq, the, thi, dt, nsub=nsub, vol=vol, coulomb_mode=oracle.COULOMB_OFF, want_cell_lum=True)
    yield "implicit", oracle.step_implicit(tab, un, rho, bsq, the, thi, dt, nsub=nsub, vol=vol, coulomb_mode=oracle.COULOMB_OFF, want_cell_lum=True)


@pytest.mark.parametrize("nsub", [1, 3])
def test_luminosity_split_single_process_limits(oracle, nsub):
    """(i) no synchrotron (Q_syn = 1e-300, eta = 1): everything is bremsstrahlung; (ii) no bremsstrahlung, eta = 1:
    everything is synchrotron, nothing Compton; (iii) no bremsstrahlung, eta = 3: Compton-added = (eta - 1) x synchrotron
    = exactly twice the synchrotron share.  A swap of two shares, or shares of anything but Q_thin, fails one of these."""
    un = oracle.Units()
    rho, bsq, the, thi = _cells(400, seed=41)
    vol = np.random.default_rng(42).uniform(0.5, 2.0, rho.size)
    dt = 3.0
    for name, o in _both_schemes(oracle, _proc_table(oracle, -9.0, -300.0, 0.0), un, rho, bsq, the, thi, dt, vol, nsub):
        d = o["diag"]
        assert d["lum_total"] > 0 and d["lum_brems"] == pytest.approx(d["lum_total"], rel=1e-14), name
        assert d["lum_synch"] <= 1e-250 * d["lum_total"] and d["lum_compton"] == 0.0, name
        assert o["cell_lum"][:, 1] == pytest.approx(o["cell_lum"][:, 0], rel=1e-14)
    for name, o in _both_schemes(oracle, _proc_table(oracle, -300.0, -9.0, 0.0), un, rho, bsq, the, thi, dt, vol, nsub):
        d = o["diag"]
        assert d["lum_total"] > 0 and d["lum_synch"] == pytest.approx(d["lum_total"], rel=1e-14), name
        assert d["lum_brems"] <= 1e-250 * d["lum_total"] and d["lum_compton"] == 0.0, name
    log3 = float(np.float32(np.log10(3.0)))
    eta = 10.0 ** log3                                          # the value the fp32 table actually holds
    for name, o in _both_schemes(oracle, _proc_table(oracle, -300.0, -9.0, log3), un, rho, bsq, the, thi, dt, vol, nsub):
        d = o["diag"]
        assert d["lum_compton"] / d["lum_synch"] == pytest.approx(eta - 1.0, rel=1e-12), name
        assert d["lum_synch"] + d["lum_compton"] == pytest.approx(d["lum_total"], rel=1e-12), name
        cl = o["cell_lum"]
        act = cl[:, 0] > 0
        assert act.sum() > 300 and cl[act, 3] / cl[act, 2] == pytest.approx(eta - 1.0, rel=1e-12)


def test_luminosity_split_ratios_survive_bridge_and_limiter(oracle):
    """With constant process tables the shares are the same for every cell, Q_brem : Q_syn : (eta - 1) Q_syn, whether
    the cell is optically thin or thick (eq 11 rescales Q_thin as a whole) and whether or not the 30 % limiter bites."""
    un = oracle.Units()
    rho, bsq, the, thi = _cells(600, seed=43)
    rho = rho * 1e3                                             # some cells optically thick (tau_sca = 2 n_e sigma_T H > 1)
    lb, ls, le = -1.0, -1.5, float(np.float32(0.25))    # strong enough for tau_abs ~ 1 in the cold cells
    qbr, qsy, eta = 10.0 ** lb, 10.0 ** ls, 10.0 ** le
    qthin = qbr + eta * qsy
    tab = _proc_table(oracle, lb, ls, le)
    for dt in (1e-12, 1e3):                                     # unlimited / mostly limited
        o = oracle.step(tab, un, rho, bsq, the, thi, dt, nsub=2, coulomb_mode=oracle.COULOMB_OFF, want_cell_lum=True, want_rates=True)
        cl = o["cell_lum"]
        assert cl[:, 1] / cl[:, 0] == pytest.approx(qbr / qthin, rel=1e-12)
        assert cl[:, 2] / cl[:, 0] == pytest.approx(qsy / qthin, rel=1e-12)
        assert cl[:, 3] / cl[:, 0] == pytest.approx((eta - 1.0) * qsy / qthin, rel=1e-12)
        # the bridge really is exercised: Q_total / Q_thin spans thin (-> 1) and thick (<< 1) cells
        ratio = o["lam0"] / qthin
        assert ratio.max() > 0.99 and ratio.min() < 0.5
    assert 0 < o["diag"]["n_limited"] <= rho.size


def test_luminosity_split_one_cell_by_hand(oracle):
    """One cell written out from eqs 10-14 with unequal shares: H_th = c_s/Omega_K (eqs 13-14),
    tau_sca = 2 n_e sigma_T H, tau_abs = H Q_thin/(4 sigma_SB T_e^4) (eq 12), Q_total of eq 11, then the shares of C-21."""
    un = oracle.Units()
    c, kB, me, mp, sigT, sigSB, GMsun = 2.99792458e10, 1.380649e-16, 9.1093837015e-28, 1.67262192369e-24, 6.6524587321e-25, 5.670374419e-5, 1.32712440018e26
    rho, bsq, the, thi, vol, dt = 2e-2, 1e-4, 0.4, 5.0, 1.7, 1e-5
    lb, ls, le = float(np.float32(-6.2)), float(np.float32(-7.1)), float(np.float32(0.6))
    tab = _proc_table(oracle, lb, ls, le)
    o = oracle.step(tab, un, np.array([rho]), np.array([bsq]), np.array([the]), np.array([thi]), dt, vol=np.array([vol]),
                    coulomb_mode=oracle.COULOMB_OFF)
    # by hand, cgs
    rg = GMsun * 10.0 / c ** 2
    tg = rg / c
    conv = tg / (3e-7 * c ** 2)                                  # erg cm^-3 s^-1 -> code units
    pe, pi = the * me / mp, thi * me / mp
    cs2 = (5.0 / 3.0) * (pe + pi) / (1.0 + 1.5 * (pe + pi) + pe + pi)          # eq 14: gamma P/(rho + u + P), u = P/(gamma-1)
    H = rg * math.sqrt(cs2) * (10.0 ** 1.5 + 0.9375)             # eq 13 at r_ref = 10 r_g: c_s / Omega_K
    ne = rho * 3e-7 / mp
    Te = the * me * c ** 2 / kB
    qbr, qsy, eta = 10.0 ** lb / conv, 10.0 ** ls / conv, 10.0 ** le
    qthin = qbr + eta * qsy                                      # eq 10
    bb = 4.0 * sigSB * Te ** 4
    tau_sca, tau_abs = 2.0 * ne * sigT * H, H * qthin / bb       # eq 12
    qtot = (bb / H) / (1.5 * (tau_abs + tau_sca) + math.sqrt(3.0) + 1.0 / tau_abs) * conv     # eq 11
    ue = rho * the * (me / mp) / (2.0 / 3.0)
    assert qtot * dt < 0.3 * ue                                  # the limiter is idle for this cell
    d = o["diag"]
    assert d["lum_total"] == pytest.approx(qtot * vol, rel=1e-12)
    assert d["lum_brems"] == pytest.approx(qtot * vol * qbr / qthin, rel=1e-12)
    assert d["lum_synch"] == pytest.approx(qtot * vol * qsy / qthin, rel=1e-12)
    assert d["lum_compton"] == pytest.approx(qtot * vol * (eta - 1.0) * qsy / qthin, rel=1e-12)
    assert len({round(d[k] / d["lum_total"], 3) for k in ("lum_brems", "lum_synch", "lum_compton")}) == 3      # unequal shares
    fr = oracle.combine_code(un, rho, the, thi, 10.0 ** lb, 10.0 ** ls, eta)[1]
    assert fr == pytest.approx([qbr / qthin, qsy / qthin, (eta - 1.0) * qsy / qthin], rel=1e-13)
