"""Pins for oracle Part C — the radiation-pressure temperature correction (eq 29; reading C-20 of
DESIGN.md).  The paper prints no worked number for it beyond "T_e ~ 1e9 K -> ~1e6 K" (L345), so the pins are
manufactured roots (exact inverse of eq 29), high-precision roots of the UNREDUCED eq 29 (with T_i on both sides) from
mpmath, both asymptotic limits, and the threshold on tau_sca = n_e sigma_T H written out by hand.  None of the expected
values comes from the oracle or the CUDA path.  CPU only."""
import numpy as np
import pytest

KB, ME, MP, CL = 1.380649e-16, 9.1093837015e-28, 1.67262192369e-24, 2.99792458e10
SIGT, GMSUN = 6.6524587321e-25, 1.32712440018e26
ARAD = 7.5646e-15                         # erg cm^-3 K^-4, as the paper prints it (L345)
TK = ME * CL * CL / KB                    # K per unit Theta


def _rg(un):
    return GMSUN * un.mbh_msun / CL ** 2


def test_manufactured_roots(oracle):
    """Pick the answer T' first: eq 29 with P = N k (T_e + T_i) gives T_e = T' + a T'^4/(N k) in closed form."""
    un = oracle.Units()
    rng = np.random.default_rng(3)
    n = 4000
    rho = 10 ** rng.uniform(-6, 0, n)
    Tnew = 10 ** rng.uniform(1.5, 8.0, n)                          # K
    N = rho * un.rho_scale_cgs / MP
    Te = Tnew + ARAD * Tnew ** 4 / (N * KB)
    hs = np.full(n, 1e30)                                          # tau_sca far above any threshold
    out, cnt = oracle.radpress(un, rho, Te / TK, hs, tau_crit=1.0)
    assert cnt == n
    assert out * TK == pytest.approx(Tnew, rel=1e-13)
    ratio = Tnew / Te                                               # both regimes are exercised
    assert (ratio < 1e-3).sum() > 200 and (ratio > 0.999).sum() > 200 and ((ratio > 0.1) & (ratio < 0.9)).sum() > 200


def test_unreduced_quartic_with_mpmath(oracle):
    """a T^4 + N k (T + T_i) = N k (T_e + T_i) solved at 60 digits with T_i kept on both sides (the oracle cancels it)."""
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 60
    un = oracle.Units()
    rng = np.random.default_rng(4)
    rho = 10 ** rng.uniform(-6, 0, 40)
    the = 10 ** rng.uniform(-3, 1.5, 40)
    thi = 10 ** rng.uniform(-3, 1.5, 40)
    out, _ = oracle.radpress(un, rho, the, np.full(40, 1e30), tau_crit=1.0)
    for k in range(40):
        N = mp.mpf(float(rho[k])) * mp.mpf(un.rho_scale_cgs) / mp.mpf(MP)
        Te, Ti = mp.mpf(float(the[k])) * mp.mpf(TK), mp.mpf(float(thi[k])) * mp.mpf(TK)
        P = N * KB * (Te + Ti)
        roots = mp.polyroots([mp.mpf(ARAD), 0, 0, N * KB, N * KB * Ti - P], maxsteps=500, extraprec=400)
        pos = [r.real for r in roots if abs(r.imag) < mp.mpf(10) ** -30 * abs(r) and r.real > 0]
        assert len(pos) == 1                                       # exactly one positive real root
        assert out[k] * TK == pytest.approx(float(pos[0]), rel=1e-13)
        assert 0 < out[k] <= the[k]


def test_limits(oracle):
    """beta = a T_e^3/(N k): beta << 1 -> T' = T_e (1 - beta + 4 beta^2 - ...); beta >> 1 -> T' = (N k T_e/a)^(1/4) (1 - y0/4 + ...)."""
    un = oracle.Units()
    rho = np.array([1.0, 0.3, 1e-2])
    N = rho * un.rho_scale_cgs / MP
    hs = np.full(3, 1e30)
    Te = np.array([1e4, 5e3, 1e3])                                  # gas-pressure dominated
    beta = ARAD * Te ** 3 / (N * KB)
    assert beta.max() < 1e-3
    out, _ = oracle.radpress(un, rho, Te / TK, hs)
    assert out * TK / Te == pytest.approx(1 - beta + 4 * beta ** 2, abs=30 * beta.max() ** 3 + 1e-15)
    Te = np.array([1e11, 3e10, 1e11])                               # radiation-pressure dominated
    beta = ARAD * Te ** 3 / (N * KB)
    assert beta.min() > 1e8
    y0 = beta ** -0.25
    out, _ = oracle.radpress(un, rho, Te / TK, hs)
    assert out * TK / Te == pytest.approx(y0 * (1 - y0 / 4), rel=2 * y0.max() ** 2)
    # the paper's orders of magnitude (L345): T_e ~ 1e9 K drops to ~1e6 K at the densities of the thick disk
    out, _ = oracle.radpress(un, np.array([1.0]), np.array([1e9 / TK]), np.array([1e30]))
    assert 3e5 < out[0] * TK < 3e7


def test_threshold_and_passthrough(oracle):
    un = oracle.Units()
    rng = np.random.default_rng(8)
    n = 2000
    rho = 10 ** rng.uniform(-6, 0, n)
    the = 10 ** rng.uniform(-3, 1.5, n)
    hs = rng.uniform(0.05, 30.0, n)                                 # scale height in r_g
    tau = rho * un.rho_scale_cgs / MP * SIGT * hs * _rg(un)         # L353, by hand
    assert oracle.tau_sca(un, float(rho[0]), float(hs[0])) == pytest.approx(tau[0], rel=1e-14)
    for crit in (1.0, 4.6):
        out, cnt = oracle.radpress(un, rho, the, hs, tau_crit=crit)
        thick = tau > crit
        assert 0 < thick.sum() < n and cnt == thick.sum()
        assert np.array_equal(out[~thick], the[~thick])             # thin cells untouched, bit for bit
        assert (out[thick] < the[thick]).all() and (out[thick] > 0).all()
    # rho <= 0, Theta_e <= 0 and NaN pass through
    rho2, the2 = rho.copy(), the.copy()
    rho2[3] = 0.0; the2[4] = -1.0; the2[5] = np.nan
    out, _ = oracle.radpress(un, rho2, the2, np.full(n, 1e30))
    assert out[3] == the2[3] and out[4] == -1.0 and np.isnan(out[5])
    # a larger threshold corrects a subset; raising density at fixed T_e lowers beta, so T'/T_e rises
    o1, _ = oracle.radpress(un, np.array([1e-3, 1e-2, 1e-1]), np.full(3, 0.2), np.full(3, 1e30))
    assert o1[0] < o1[1] < o1[2] < 0.2
