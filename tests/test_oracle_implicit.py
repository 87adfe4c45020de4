"""Pins for oracle Part B' — the implicit scheme (PAPER.md L185 (ii), L369; reading C-18 of DESIGN.md: backward Euler
for the radiative sink with the cooling time held outside the table's Theta_e range, Coulomb coefficient at the start
state and driving difference at the end state).  The paper gives no equations and prints no numbers for it, so the pins
are closed forms of special cases, limits and invariants; none is produced by the oracle or the CUDA path.  CPU only."""
import numpy as np
import pytest

ME, MP = 9.1093837015e-28, 1.67262192369e-24
MR = ME / MP
GE1 = GI1 = 2.0 / 3.0
LO3, HI3 = [-6.0, -3.0, -8.0], [0.0, 1.5, 0.0]


def _cells(n, seed=5, the_range=(-3, 1.5)):
    rng = np.random.default_rng(seed)
    return (10 ** rng.uniform(-6, 0, n), 10 ** rng.uniform(-8, 0, n),
            10 ** rng.uniform(*the_range, n), 10 ** rng.uniform(-3, 1.5, n))


def _const_lambda_table(oracle, log_lambda, coul_logC=None):
    data = [np.full((3, 3, 3), log_lambda, dtype=np.float32)]
    kw = {} if coul_logC is None else dict(coul=np.full((3, 3), coul_logC, np.float32), clo=[-3.0, -3.0], chi=[1.5, 1.5])
    return oracle.Table([0, 1, 2], [3, 3, 3], LO3, HI3, data, **kw)


def _const_tcool_table(oracle, c0):
    """log10 Lambda = c0 + log10 rho + log10 Theta_e on integer nodes (exact in fp32, exact under multilinear
    interpolation): Lambda = 10^c0 rho Theta_e, i.e. a constant cooling time."""
    lo, hi, n = [-6.0, -3.0, -8.0], [0.0, 2.0, 0.0], [7, 6, 3]
    xr, xe, _ = np.meshgrid(np.linspace(lo[0], hi[0], n[0]), np.linspace(lo[1], hi[1], n[1]), np.linspace(lo[2], hi[2], n[2]), indexing="ij")
    return oracle.Table([0, 1, 2], n, lo, hi, [(c0 + xr + xe).astype(np.float32)])


def test_constant_cooling_time_closed_form(oracle):
    """Lambda = K rho Theta_e  =>  dTheta_e/dt = -Theta_e/t_c with t_c = MR/(K ge1): backward Euler gives
    Theta_e' = Theta_e/(1 + h/t_c) per sub-step, also outside the Theta_e range (cooling time held at the edge)."""
    un = oracle.Units()
    c0 = -5.0
    tc = MR / (10.0 ** c0 * GE1)
    tab = _const_tcool_table(oracle, c0)
    rho, bsq, the, thi = _cells(400, the_range=(-4.5, 3.0))          # includes cells below and above the table's Theta_e range
    for dt, nsub in ((0.3 * tc, 1), (50.0 * tc, 1), (1e4 * tc, 3)):
        o = oracle.step_implicit(tab, un, rho, bsq, the, thi, dt, nsub=nsub, coulomb_mode=oracle.COULOMB_OFF)
        h = dt / nsub
        assert o["theta_e"] == pytest.approx(the / (1.0 + h / tc) ** nsub, rel=1e-12)
        assert np.array_equal(o["theta_i"], thi)
        assert (o["theta_e"] > 0).all()


def test_constant_lambda_piecewise_closed_form(oracle):
    """Constant Lambda inside the table: backward Euler = forward Euler, Theta_e' = Theta_e - h Lambda k while that
    stays above the lower Theta_e edge; below it the cooling time is held, Theta_e' = Theta_e/(1 + h Lambda k/theta_min).
    k = ge1/(MR rho).  Never negative however large h Lambda is (the explicit scheme needs the 30 % limiter for that)."""
    un = oracle.Units()
    lam = 1e-9
    tab = _const_lambda_table(oracle, -9.0)
    rho, bsq, the, thi = _cells(3000, seed=9)
    the = np.clip(the, 1e-3, 10 ** 1.5)
    tmin = 1e-3
    for dt in (1e-3, 1.0, 1e3, 1e6):
        o = oracle.step_implicit(tab, un, rho, bsq, the, thi, dt, coulomb_mode=oracle.COULOMB_OFF)
        drop = dt * lam * GE1 / (MR * rho)
        inside = the - drop >= tmin
        ref = np.where(inside, the - drop, the / (1.0 + drop / tmin))
        assert o["theta_e"] == pytest.approx(ref, rel=1e-11)
        assert (o["theta_e"] > 0).all()
        if dt >= 1e3:
            assert (~inside).sum() > 100 and inside.sum() > 0          # both branches exercised
        # diagnostic = radiated energy / dt
        lost = rho * (the - o["theta_e"]) * MR / GE1
        assert o["diag"]["lum_total"] == pytest.approx(float(lost.sum() / dt), rel=1e-9)
        assert o["diag"]["n_limited"] == 0


def test_coulomb_only_closed_form(oracle):
    """Negligible Lambda, constant C: the sub-step is the linear backward-Euler relaxation
    theta' = (Theta_e (1 + a g) + a Theta_i)/(1 + a g + a), Theta_i' = Theta_i - g a (Theta_i - theta')/(1 + a g).
    K is written out from eq 15 (L142-L144) with the prefactor (3/2)(m_e/m_p) ln(Lambda) c sigma_T m_e c^2 =
    2.667753872e-22 erg cm^3/s (SURVEY 8(c) pin): dTheta_e/dt = K C (Theta_i - Theta_e),
    K = 2.667753872e-22 (rho_scale/m_p)^2 rho t_g/(rho_scale c^2) (gamma_e - 1)/(m_e/m_p)."""
    un = oracle.Units()
    logC = 0.5
    tab = _const_lambda_table(oracle, -37.0, coul_logC=logC)
    rho, bsq, the, thi = _cells(500, seed=3)
    c_cgs, tg = 2.99792458e10, 1.32712440018e26 * un.mbh_msun / 2.99792458e10 ** 3
    KC = 2.667753872e-22 * (un.rho_scale_cgs / MP) ** 2 * rho * tg / (un.rho_scale_cgs * c_cgs ** 2) * GE1 / MR * 10.0 ** logC
    ok = np.ones(rho.size, bool)
    g = GI1 / GE1
    for dt, nsub in ((1e-2, 1), (1e3, 1), (1e7, 2)):
        o = oracle.step_implicit(tab, un, rho, bsq, the, thi, dt, nsub=nsub)
        te, ti = the.copy(), thi.copy()
        for _ in range(nsub):
            a = dt / nsub * KC
            tn = (te * (1 + a * g) + a * ti) / (1 + a * g + a)
            ti = ti - g * a * (ti - tn) / (1 + a * g)
            te = tn
        assert o["theta_e"][ok] == pytest.approx(te[ok], rel=1e-9)     # 2.667753872e-22 carries 10 digits
        assert o["theta_i"][ok] == pytest.approx(ti[ok], rel=1e-9)
        # exact invariants: energy conserved, no crossing, relaxation towards each other
        tot0, tot1 = the / GE1 + thi / GI1, o["theta_e"] / GE1 + o["theta_i"] / GI1
        assert tot1 == pytest.approx(tot0, rel=1e-12)
        assert (np.sign(o["theta_i"] - o["theta_e"]) * np.sign(thi - the) >= 0).all()
        assert (np.abs(o["theta_i"] - o["theta_e"]) <= np.abs(thi - the) * (1 + 1e-12)).all()
    # equal temperatures stay equal (zero exchange at T_e = T_i)
    o = oracle.step_implicit(tab, un, rho, bsq, the, the, 1e3)
    assert o["theta_e"] == pytest.approx(the, rel=1e-14) and o["theta_i"] == pytest.approx(the, rel=1e-14)


def test_small_dt_matches_unlimited_explicit_and_root_residual(oracle):
    """Small changes: implicit and (unlimited) explicit updates differ at second order; F(theta') = 0 to rounding on a rough table."""
    un = oracle.Units()
    rng = np.random.default_rng(11)
    n = [6, 7, 5]
    T = rng.uniform(-12.0, -6.0, size=n).astype(np.float32)
    C = rng.uniform(-1.0, 1.0, size=(4, 5)).astype(np.float32)
    tab = oracle.Table([0, 1, 2], n, LO3, HI3, [T], coul=C, clo=[-3.0, -3.0], chi=[1.5, 1.5])
    rho, bsq, the, thi = _cells(800, seed=12)
    # consistency: where the explicit step is not limited, the two schemes differ only at second order in the change,
    # |implicit - explicit| <= K change^2/Theta (K bounded by the table's logarithmic slope), and really do differ
    for dt in (1e-2, 1e-4):
        e = oracle.step(tab, un, rho, bsq, the, thi, dt, f_limit=0.49, want_rates=True)
        i = oracle.step_implicit(tab, un, rho, bsq, the, thi, dt)
        ch = np.abs(e["theta_e"] - the) + np.abs(e["theta_i"] - thi)
        small = ch < 1e-2 * np.minimum(the, thi)
        diff = np.abs(i["theta_e"] - e["theta_e"])
        second = ch * ch / np.minimum(the, thi)
        assert small.sum() > 400
        assert (diff[small] <= 100.0 * second[small] + 1e-14 * the[small]).all()
        probe = small & (ch > 1e-4 * np.minimum(the, thi))
        assert probe.sum() > 20 and np.median(diff[probe] / second[probe]) > 1e-3
    dt = 30.0
    o = oracle.step_implicit(tab, un, rho, bsq, the, thi, dt)
    for k in range(0, 800, 7):
        F = oracle.implicit_residual(tab, un, rho[k], bsq[k], the[k], thi[k], dt, o["theta_e"][k])
        assert abs(F) <= 1e-12 * max(the[k], o["theta_e"][k], thi[k])
    assert (o["theta_e"] > 0).all() and (o["theta_i"] > 0).all()
    # energy leaves only through radiation
    lost = rho * ((the + thi) - (o["theta_e"] + o["theta_i"])) * MR / GE1
    assert o["diag"]["lum_total"] == pytest.approx(float(lost.sum() / dt), rel=1e-9)


def test_four_d_tables_and_floor(oracle):
    """nproc = 3 tables (eqs 10-14 with H from the trial Theta_e and the start Theta_i), floor flag, luminosity split."""
    un = oracle.Units()
    rng = np.random.default_rng(21)
    n = [4, 5, 3, 4]
    lo, hi = LO3 + [-3.0], HI3 + [1.5]
    data = [rng.uniform(-14.0, -8.0, size=n).astype(np.float32), rng.uniform(-14.0, -8.0, size=n).astype(np.float32),
            rng.uniform(0.0, 1.0, size=n).astype(np.float32)]
    tab = oracle.Table([0, 1, 2, 3], n, lo, hi, data, coul=np.zeros((3, 3), np.float32), clo=[-3.0, -3.0], chi=[1.5, 1.5])
    rho, bsq, the, thi = _cells(600, seed=22)
    r = np.random.default_rng(23).uniform(2.0, 50.0, rho.size)
    o = oracle.step_implicit(tab, un, rho, bsq, the, thi, 100.0, nsub=2, h_floor=0.1, r=r)
    d = o["diag"]
    assert 0 < d["n_floored"] < rho.size
    assert d["lum_brems"] + d["lum_synch"] + d["lum_compton"] == pytest.approx(d["lum_total"], rel=1e-12)
    lost = rho * ((the + thi) - (o["theta_e"] + o["theta_i"])) * MR / GE1
    assert d["lum_total"] == pytest.approx(float(lost.sum() / 100.0), rel=1e-9)
    assert (o["theta_e"] > 0).all() and (o["theta_i"] > 0).all()
    # NaN in -> NaN out for that cell only; rho <= 0 passes through
    the2 = the.copy(); the2[5] = np.nan; rho2 = rho.copy(); rho2[7] = 0.0
    o2 = oracle.step_implicit(tab, un, rho2, bsq, the2, thi, 100.0, nsub=2)
    assert np.isnan(o2["theta_e"][5]) and np.isnan(o2["theta_i"][5]) and o2["theta_e"][7] == the[7] and o2["theta_i"][7] == thi[7]
    assert np.isfinite(np.delete(o2["theta_e"], 5)).all()
