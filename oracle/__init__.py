"""ORACLE — test infrastructure, NOT the product.

Thin ctypes/numpy front end of ``oracle/cool_oracle.c`` (plain fp64 C statement of the
cooling step of arXiv 2505.08855; see that file's header for the passages it follows).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2505_08855_b200`` and the product imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cool_oracle.c")
_LIB = os.path.join(_HERE, "libcool_oracle.so")

AX_LOG_RHO, AX_LOG_THETA_E, AX_LOG_BSQ, AX_LOG_THETA_I = 0, 1, 2, 3
AX_LOG_HTH, AX_LOG_B, AX_LOG_NE, AX_LOG_TE = 4, 5, 6, 7           # Part D: the paper's parameters in cgs units


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (no fast-math).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Units(C.Structure):
    """Mirror of ``orc_units``; defaults follow SURVEY §8(d) (EXP_HIGH rho_scale)."""
    _fields_ = [(n, C.c_double) for n in (
        "rho_scale_cgs", "mbh_msun", "gamma_e", "gamma_i", "ln_lambda",
        "ion_theta_mass_ratio", "hth_cm", "r_ref_rg", "spin")]

    def __init__(self, rho_scale_cgs=3e-7, mbh_msun=10.0, gamma_e=5.0 / 3.0, gamma_i=5.0 / 3.0,
                 ln_lambda=20.0, ion_theta_mass_ratio=1.0, hth_cm=1.476625e7, r_ref_rg=10.0,
                 spin=0.9375):
        super().__init__(rho_scale_cgs, mbh_msun, gamma_e, gamma_i, ln_lambda,
                         ion_theta_mass_ratio, hth_cm, r_ref_rg, spin)


class _Table(C.Structure):
    _fields_ = [("ndim", C.c_int), ("axis", C.c_int * 4), ("n", C.c_int * 4),
                ("lo", C.c_double * 4), ("hi", C.c_double * 4), ("nproc", C.c_int),
                ("data", C.POINTER(C.c_float) * 3), ("coul", C.POINTER(C.c_float)),
                ("nc", C.c_int * 2), ("clo", C.c_double * 2), ("chi", C.c_double * 2),
                ("cgs", C.c_int), ("coul3", C.POINTER(C.c_float)), ("nc3", C.c_int * 3), ("c3lo", C.c_double * 3), ("c3hi", C.c_double * 3)]


class Table:
    """A cooling table as data: ``data`` is a list of 1 or 3 float32 arrays of shape ``n``
    (row-major, last axis fastest, log10 values); ``coul`` an optional float32 (nc0, nc1)
    array of log10 C over (log Theta_i, log Theta_e)."""

    def __init__(self, axis, n, lo, hi, data, coul=None, clo=None, chi=None, cgs=False, coul3=None, c3lo=None, c3hi=None):
        """``cgs``: data[0] is the paper's table, log10 Q_total[erg cm^-3 s^-1] over (log H_th, log B, log n_e, log T_e[K]);
        ``coul3``: optional float32 (n0, n1, n2) array of log10 [Q_cc/(T_i - T_e)] over (log n_e, log T_i[K], log T_e[K])."""
        self.axis = list(axis); self.n = list(n); self.lo = list(lo); self.hi = list(hi)
        self.ndim = len(self.n)
        self.data = [np.ascontiguousarray(d, dtype=np.float32).reshape(self.n) for d in data]
        self.nproc = len(self.data)
        assert self.nproc in (1, 3)
        self.coul = None if coul is None else np.ascontiguousarray(coul, dtype=np.float32)
        self.clo = list(clo) if clo is not None else [0.0, 0.0]
        self.chi = list(chi) if chi is not None else [1.0, 1.0]
        t = _Table()
        t.ndim = self.ndim
        for k in range(self.ndim):
            t.axis[k] = self.axis[k]; t.n[k] = self.n[k]; t.lo[k] = self.lo[k]; t.hi[k] = self.hi[k]
        t.nproc = self.nproc
        for p, d in enumerate(self.data):
            t.data[p] = d.ctypes.data_as(C.POINTER(C.c_float))
        if self.coul is not None:
            t.coul = self.coul.ctypes.data_as(C.POINTER(C.c_float))
            t.nc[0], t.nc[1] = self.coul.shape
            t.clo[0], t.clo[1] = self.clo; t.chi[0], t.chi[1] = self.chi
        t.cgs = int(bool(cgs))
        self.cgs = bool(cgs)
        self.coul3 = None if coul3 is None else np.ascontiguousarray(coul3, dtype=np.float32)
        if self.coul3 is not None:
            t.coul3 = self.coul3.ctypes.data_as(C.POINTER(C.c_float))
            for k in range(3):
                t.nc3[k] = self.coul3.shape[k]; t.c3lo[k] = float(c3lo[k]); t.c3hi[k] = float(c3hi[k])
        self._c = t


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        d, i, p = C.c_double, C.c_int, C.c_void_p
        UP = C.POINTER(Units)
        sig = {
            "orc_ne_cgs": (d, [UP, d]), "orc_bfield_gauss": (d, [UP, d]),
            "orc_brems_cgs": (d, [d, d]),
            "orc_bessel_k_scaled": (d, [d, d]), "orc_bessel_k2_scaled": (d, [d]),
            "orc_iprime": (d, [d]), "orc_k2_tilde": (d, [d]),
            "orc_synch_xc": (d, [d, d, d, d]), "orc_synch_J": (d, [d]),
            "orc_synch_cgs": (d, [d, d, d, d, C.POINTER(d)]),
            "orc_compton_eta": (d, [d, d, d, d]), "orc_compton_eta_ex": (d, [d, d, d, d, i]),
            "orc_bridge_cgs": (d, [d, d, d, d]),
            "orc_cooling_cgs": (None, [d, d, d, d, C.POINTER(d)]),
            "orc_omega_k": (d, [d, d]), "orc_hth_cm": (d, [UP, d, d, d]),
            "orc_coulomb_C": (d, [d, d]), "orc_coulomb_pref_cgs": (d, [UP]),
            "orc_coulomb_code": (d, [UP, d, d, d]),
            "orc_node_total_log10": (d, [UP, d, d, d]),
            "orc_node_proc_log10": (None, [UP, d, d, d, d, C.POINTER(d)]),
            "orc_combine_code": (d, [UP, d, d, d, d, d, d, C.POINTER(d)]),
            "orc_interp": (d, [i, C.POINTER(i), C.POINTER(d), C.POINTER(d), C.POINTER(C.c_float),
                               C.POINTER(d), C.POINTER(i)]),
            "orc_step": (None, [C.POINTER(_Table), UP, C.c_longlong, p, p, p, p, p, p,
                                d, i, d, d, i, i, p, p, p, p, p, p, i, p]),
            "orc_step_implicit": (None, [C.POINTER(_Table), UP, C.c_longlong, p, p, p, p, p, p,
                                         d, i, d, i, p, p, p, p, i]),
            "orc_implicit_residual": (d, [C.POINTER(_Table), UP, d, d, d, d, d, d, i, d, i, d]),
            "orc_fill_total3": (None, [UP, C.POINTER(i), C.POINTER(d), C.POINTER(d), p, i]),
            "orc_fill_coulomb2": (None, [UP, C.POINTER(i), C.POINTER(d), C.POINTER(d), p]),
            "orc_fill_proc4": (None, [UP, C.POINTER(i), C.POINTER(d), C.POINTER(d), p, p, p, i]),
            "orc_max_threads": (i, []),
            "orc_fill_total4_cgs": (None, [C.POINTER(i), C.POINTER(d), C.POINTER(d), p, i]),
            "orc_fill_coulomb3_cgs": (None, [UP, C.POINTER(i), C.POINTER(d), C.POINTER(d), p]),
            "orc_tau_sca_cell": (d, [UP, d, d]),
            "orc_radpress": (None, [UP, C.c_longlong, p, p, p, d, p, C.POINTER(C.c_longlong)]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name); f.restype = res; f.argtypes = args
        _lib = L
    return _lib


# ---- Part A convenience wrappers (scalar in, scalar out) ---------------------------------

def brems_cgs(ne, th): return lib().orc_brems_cgs(ne, th)
def bessel_k_scaled(nu, x): return lib().orc_bessel_k_scaled(nu, x)
def bessel_k2_scaled(x): return lib().orc_bessel_k2_scaled(x)
def iprime(x): return lib().orc_iprime(x)
def k2_tilde(th): return lib().orc_k2_tilde(th)
def synch_xc(H, B, ne, th): return lib().orc_synch_xc(H, B, ne, th)
def synch_J(xc): return lib().orc_synch_J(xc)
def compton_eta(nu_c, ne, H, th, printed_exponent=False):
    return lib().orc_compton_eta_ex(nu_c, ne, H, th, int(printed_exponent))
def bridge_cgs(H, ne, th, qthin): return lib().orc_bridge_cgs(H, ne, th, qthin)
def omega_k(r, a): return lib().orc_omega_k(r, a)
def hth_cm(un, th_e, th_i, r): return lib().orc_hth_cm(C.byref(un), th_e, th_i, r)
def coulomb_C(th_e, th_i): return lib().orc_coulomb_C(th_e, th_i)
def coulomb_pref_cgs(un): return lib().orc_coulomb_pref_cgs(C.byref(un))
def coulomb_code(un, rho, th_e, th_i): return lib().orc_coulomb_code(C.byref(un), rho, th_e, th_i)
def ne_cgs(un, rho): return lib().orc_ne_cgs(C.byref(un), rho)
def bfield_gauss(un, bsq): return lib().orc_bfield_gauss(C.byref(un), bsq)
def node_total_log10(un, rho, th_e, bsq): return lib().orc_node_total_log10(C.byref(un), rho, th_e, bsq)


def synch_cgs(H, B, ne, th):
    """(Q_syn, nu_c)"""
    nuc = C.c_double()
    q = lib().orc_synch_cgs(H, B, ne, th, C.byref(nuc))
    return q, nuc.value


def cooling_cgs(H, B, ne, th):
    """dict of Q_brem, Q_syn, eta, Q_thin, Q_total [erg cm^-3 s^-1] and nu_c [Hz]."""
    out = (C.c_double * 6)()
    lib().orc_cooling_cgs(H, B, ne, th, out)
    return dict(zip(("brems", "synch", "eta", "thin", "total", "nu_c"), list(out)))


def node_proc_log10(un, rho, th_e, bsq, th_i):
    out = (C.c_double * 3)()
    lib().orc_node_proc_log10(C.byref(un), rho, th_e, bsq, th_i, out)
    return list(out)


def combine_code(un, rho, th_e, th_i, qbr, qsy, eta):
    fr = (C.c_double * 3)()
    q = lib().orc_combine_code(C.byref(un), rho, th_e, th_i, qbr, qsy, eta, fr)
    return q, list(fr)


def interp(n, lo, hi, T, x):
    """Multilinear interpolation of float32 table T (shape n) at log-coordinates x.
    Returns (y, clamped)."""
    nd = len(n)
    T = np.ascontiguousarray(T, dtype=np.float32)
    cl = C.c_int()
    y = lib().orc_interp(nd, (C.c_int * nd)(*n), (C.c_double * nd)(*lo), (C.c_double * nd)(*hi),
                         T.ctypes.data_as(C.POINTER(C.c_float)), (C.c_double * nd)(*x), C.byref(cl))
    return y, bool(cl.value)


def fill_total3(un, n, lo, hi, nthreads=0):
    out = np.empty(n, dtype=np.float32)
    lib().orc_fill_total3(C.byref(un), (C.c_int * 3)(*n), (C.c_double * 3)(*lo), (C.c_double * 3)(*hi),
                          out.ctypes.data, nthreads or max_threads())
    return out


def fill_proc4(un, n, lo, hi, nthreads=0):
    """[log10 Q_brem, log10 Q_syn, log10 eta] over (log rho, log Theta_e, log bsq, log Theta_i) from Part A."""
    outs = [np.empty(n, dtype=np.float32) for _ in range(3)]
    lib().orc_fill_proc4(C.byref(un), (C.c_int * 4)(*n), (C.c_double * 4)(*lo), (C.c_double * 4)(*hi),
                         outs[0].ctypes.data, outs[1].ctypes.data, outs[2].ctypes.data, nthreads or max_threads())
    return outs


def fill_coulomb2(un, nc, clo, chi):
    out = np.empty(nc, dtype=np.float32)
    lib().orc_fill_coulomb2(C.byref(un), (C.c_int * 2)(*nc), (C.c_double * 2)(*clo), (C.c_double * 2)(*chi),
                            out.ctypes.data)
    return out


def fill_total4_cgs(n, lo, hi, nthreads=0):
    """The paper's table (L124) from Part A: log10 Q_total[cgs] over (log H_th, log B, log n_e, log T_e[K])."""
    out = np.empty(n, dtype=np.float32)
    lib().orc_fill_total4_cgs((C.c_int * 4)(*n), (C.c_double * 4)(*lo), (C.c_double * 4)(*hi), out.ctypes.data, nthreads or max_threads())
    return out


def fill_coulomb3_cgs(un, n, lo, hi):
    """The paper's Coulomb table (L147): log10 [Q_cc/(T_i - T_e)] over (log n_e, log T_i[K], log T_e[K])."""
    out = np.empty(n, dtype=np.float32)
    lib().orc_fill_coulomb3_cgs(C.byref(un), (C.c_int * 3)(*n), (C.c_double * 3)(*lo), (C.c_double * 3)(*hi), out.ctypes.data)
    return out


def max_threads():
    n = lib().orc_max_threads()
    try:
        n = min(n, len(os.sched_getaffinity(0)))
    except AttributeError:
        pass
    return max(1, n)


RATE_TABLE, RATE_ANALYTIC = 0, 1
COULOMB_OFF, COULOMB_TABLE, COULOMB_ANALYTIC, COULOMB_TABLE3 = 0, 1, 2, 3


def step(table: Table, un: Units, rho, bsq, theta_e, theta_i, dt, nsub=1, f_limit=0.3,
         h_floor=0.0, r=None, vol=None, rate_mode=RATE_TABLE, coulomb_mode=None, nthreads=1,
         want_rates=False, want_cell_lum=False, want_cell_flags=False):
    """Part B over a field.  Inputs are converted to float64 exactly (float32 inputs are
    representable).  Returns dict(theta_e, theta_i, diag[, lam0, qcc0])."""
    f64 = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float64).ravel()
    rho, bsq, the, thi, r, vol = map(f64, (rho, bsq, theta_e, theta_i, r, vol))
    n = rho.size
    if coulomb_mode is None:
        coulomb_mode = COULOMB_TABLE3 if table.coul3 is not None else (COULOMB_TABLE if table.coul is not None else COULOMB_ANALYTIC)
    if coulomb_mode == COULOMB_TABLE:
        assert table.coul is not None
    if coulomb_mode == COULOMB_TABLE3:
        assert table.coul3 is not None
    the_o = np.empty(n); thi_o = np.empty(n)
    lam0 = np.empty(n) if want_rates else None
    qcc0 = np.empty(n) if want_rates else None
    diag = np.zeros(7)
    cell_lum = np.zeros((n, 4)) if want_cell_lum else None
    cell_flags = np.zeros(n, dtype=np.uint8) if want_cell_flags else None
    ptr = lambda a: None if a is None else a.ctypes.data
    lib().orc_step(C.byref(table._c), C.byref(un), n, ptr(rho), ptr(bsq), ptr(the), ptr(thi),
                   ptr(r), ptr(vol), float(dt), int(nsub), float(f_limit), float(h_floor),
                   int(rate_mode), int(coulomb_mode), ptr(the_o), ptr(thi_o), ptr(lam0), ptr(qcc0),
                   ptr(cell_lum), ptr(diag), int(nthreads), ptr(cell_flags))
    out = dict(theta_e=the_o, theta_i=thi_o,
               diag=dict(lum_total=diag[0], lum_brems=diag[1], lum_synch=diag[2], lum_compton=diag[3],
                         n_limited=int(diag[4]), n_floored=int(diag[5]), n_clamped=int(diag[6])))
    if want_rates:
        out["lam0"] = lam0; out["qcc0"] = qcc0
    if want_cell_lum:
        out["cell_lum"] = cell_lum
    if want_cell_flags:
        out["cell_flags"] = cell_flags            # bit 0 limited, bit 1 floored, bit 2 clamped (per-cell terms of the counts)
    return out


def step_implicit(table: Table, un: Units, rho, bsq, theta_e, theta_i, dt, nsub=1, h_floor=0.0, r=None, vol=None,
                  coulomb_mode=None, nthreads=1, want_cell_lum=False):
    """Part B' (implicit scheme, PAPER.md L185 (ii), reading C-18) over a field.  Returns dict(theta_e, theta_i, diag)."""
    f64 = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float64).ravel()
    rho, bsq, the, thi, r, vol = map(f64, (rho, bsq, theta_e, theta_i, r, vol))
    n = rho.size
    assert not table.cgs, "the implicit scheme is not defined on the paper's cgs table here"
    if coulomb_mode is None:
        coulomb_mode = COULOMB_TABLE if table.coul is not None else COULOMB_ANALYTIC
    the_o = np.empty(n); thi_o = np.empty(n)
    diag = np.zeros(7)
    cell_lum = np.zeros((n, 4)) if want_cell_lum else None
    ptr = lambda a: None if a is None else a.ctypes.data
    lib().orc_step_implicit(C.byref(table._c), C.byref(un), n, ptr(rho), ptr(bsq), ptr(the), ptr(thi), ptr(r), ptr(vol),
                            float(dt), int(nsub), float(h_floor), int(coulomb_mode), ptr(the_o), ptr(thi_o), ptr(cell_lum),
                            ptr(diag), int(nthreads))
    out = dict(theta_e=the_o, theta_i=thi_o,
               diag=dict(lum_total=diag[0], lum_brems=diag[1], lum_synch=diag[2], lum_compton=diag[3],
                         n_limited=int(diag[4]), n_floored=int(diag[5]), n_clamped=int(diag[6])))
    if want_cell_lum:
        out["cell_lum"] = cell_lum
    return out


def shell_sums(cell_lum, shell_cells):
    """Radial luminosity profile (eq 25, numerator): partial sums of the per-cell terms over consecutive groups of
    ``shell_cells`` cells (one radial shell = all (theta, phi) cells of one r index; phi fastest)."""
    n = cell_lum.shape[0]
    starts = np.arange(0, n, int(shell_cells))
    return np.add.reduceat(cell_lum, starts, axis=0)


def implicit_residual(table: Table, un: Units, rho, bsq, theta_e, theta_i, dt, theta_trial, nsub=1, h_floor=0.0, r=0.0,
                      coulomb_mode=None):
    """F(theta_trial) of the first implicit sub-step of one cell (0 at a root)."""
    if coulomb_mode is None:
        coulomb_mode = COULOMB_TABLE if table.coul is not None else COULOMB_ANALYTIC
    return lib().orc_implicit_residual(C.byref(table._c), C.byref(un), float(rho), float(bsq), float(theta_e), float(theta_i),
                                       float(r), float(dt), int(nsub), float(h_floor), int(coulomb_mode), float(theta_trial))


# ---- Part C: radiation-pressure temperature correction (eq 29) ---------------------------
def tau_sca(un, rho, hscale_rg): return lib().orc_tau_sca_cell(C.byref(un), rho, hscale_rg)


def radpress(un: Units, rho, theta_e, hscale_rg, tau_crit=1.0):
    """Theta_e corrected for radiation pressure where tau_sca = n_e sigma_T H > tau_crit (eq 29; C-20).
    Returns (theta_e_out, n_corrected)."""
    rho, the, hs = (np.ascontiguousarray(a, dtype=np.float64) for a in (rho, theta_e, hscale_rg))
    out = np.empty_like(the)
    cnt = C.c_longlong(0)
    lib().orc_radpress(C.byref(un), rho.size, rho.ctypes.data, the.ctypes.data, hs.ctypes.data, float(tau_crit),
                       out.ctypes.data, C.byref(cnt))
    return out, int(cnt.value)
