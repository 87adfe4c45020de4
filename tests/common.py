"""Shared helpers of the test-suite: table construction (product builder -> same fp32 arrays to
the oracle: the table is data), GPU runs through the Python binding of the C ABI, comparisons."""
from __future__ import annotations

import ctypes as C

import numpy as np

from paper_2505_08855_b200 import api, synth

LO3 = [synth.LOG_RHO[0], synth.LOG_THETA[0], synth.LOG_BSQ[0]]
HI3 = [synth.LOG_RHO[1], synth.LOG_THETA[1], synth.LOG_BSQ[1]]
LO4 = LO3 + [synth.LOG_THETA[0]]
HI4 = HI3 + [synth.LOG_THETA[1]]
CLO = [synth.LOG_THETA[0]] * 2
CHI = [synth.LOG_THETA[1]] * 2

_cache = {}


def build_tables(n, nc=None, units_kw=None, axis=None, lo=None, hi=None):
    """Build (desc, data, coul) with the product's host builder; cached per shape."""
    key = (tuple(n), None if nc is None else tuple(nc), tuple(sorted((units_kw or {}).items())),
           None if axis is None else tuple(axis), None if lo is None else tuple(lo), None if hi is None else tuple(hi))
    if key not in _cache:
        nd = len(n)
        axis = list(range(nd)) if axis is None else list(axis)
        rng = {0: synth.LOG_RHO, 1: synth.LOG_THETA, 2: synth.LOG_BSQ, 3: synth.LOG_THETA}   # by cool_axis kind
        lo = [rng[a][0] for a in axis] if lo is None else list(lo)
        hi = [rng[a][1] for a in axis] if hi is None else list(hi)
        desc = api.make_desc(axis, n, lo, hi, 1 if nd == 3 else 3, units=api.default_units(**(units_kw or {})),
                             nc=nc, clo=CLO if nc else None, chi=CHI if nc else None)
        data, coul = api.cool_table_build_host(desc, want_coulomb=nc is not None)
        _cache[key] = (desc, data, coul)
    return _cache[key]


def oracle_units(oracle, desc):
    u = desc.units
    return oracle.Units(u.rho_scale_cgs, u.mbh_msun, u.gamma_e, u.gamma_i, u.ln_lambda,
                        u.ion_theta_mass_ratio, u.hth_cm, u.r_ref_rg, u.spin)


def oracle_table(oracle, desc, data, coul):
    nd = desc.ndim
    return oracle.Table([desc.axis[k] for k in range(nd)], [desc.n[k] for k in range(nd)],
                        [desc.lo[k] for k in range(nd)], [desc.hi[k] for k in range(nd)], data,
                        coul=coul, clo=[desc.clo[0], desc.clo[1]], chi=[desc.chi[0], desc.chi[1]])


def gpu_step(table, fields, dtype, dt, nsub=1, f_limit=0.3, h_floor=0.0, variant=api.COOL_V_AUTO,
             coulomb=api.COOL_COULOMB_AUTO, want_diag=True, use_r=False, use_vol=False, inplace=False, offset=0,
             scheme=api.COOL_SCHEME_EXPLICIT, shell_cells=0, want_flags=False):
    """One cool_apply on cuda:0 through the C ABI.  ``offset`` (elements) misaligns the arrays."""
    import torch
    tdt = torch.float32 if dtype == np.float32 else torch.float64
    cdt = api.COOL_F32 if dtype == np.float32 else api.COOL_F64
    dev = torch.device("cuda:0")

    def up(a):
        if a is None:
            return None
        t = torch.empty(a.size + offset, dtype=tdt, device=dev)
        t[offset:].copy_(torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)))
        return t[offset:]
    n = fields["rho"].size
    rho, bsq, the, thi = (up(fields[k]) for k in ("rho", "bsq", "theta_e", "theta_i"))
    r = up(fields["r"]) if use_r else None
    vol = up(fields["vol"]) if use_vol else None
    if inplace:
        the_o, thi_o = the, thi
    else:
        the_o = torch.empty(n + offset, dtype=tdt, device=dev)[offset:]
        thi_o = torch.empty(n + offset, dtype=tdt, device=dev)[offset:]
    d_diag = torch.zeros(api.DIAG_BYTES, dtype=torch.uint8, device=dev) if want_diag else None
    params = api.make_params(dt, nsub, f_limit, h_floor, variant, coulomb, scheme)
    stream = torch.cuda.current_stream().cuda_stream
    lum_shell = None
    if shell_cells:
        lum_shell = torch.full((4 * ((n + shell_cells - 1) // shell_cells),), -1.0, dtype=torch.float64, device=dev)   # must be overwritten
    flags = torch.full((n + 4,), 255, dtype=torch.uint8, device=dev)[offset % 4:][:n] if want_flags else None   # must be overwritten
    api.cool_apply(table, n, cdt, rho, bsq, the, thi, the_o, thi_o, params, r=r, vol=vol, d_diag=d_diag, stream=stream,
                   shell_cells=shell_cells, lum_shell=lum_shell, flags=flags)
    torch.cuda.synchronize()
    out = dict(theta_e=the_o.cpu().numpy().astype(np.float64), theta_i=thi_o.cpu().numpy().astype(np.float64),
               launches=api.cool_last_launch_count(), kernel=api.cool_last_kernel_name())
    if flags is not None:
        out["flags"] = flags.cpu().numpy()
    if want_diag:
        raw = d_diag.cpu().numpy().tobytes()
        out["diag"] = api.cool_diag.from_buffer_copy(raw).as_dict()
    if lum_shell is not None:
        out["lum_shell"] = lum_shell.cpu().numpy().reshape(-1, 4)
    return out


def oracle_step(oracle, otab, un, fields, dt, nsub=1, f_limit=0.3, h_floor=0.0, use_r=False, use_vol=False,
                rate_mode=0, coulomb_mode=None, nthreads=0, **kw):
    return oracle.step(otab, un, fields["rho"], fields["bsq"], fields["theta_e"], fields["theta_i"], dt, nsub=nsub,
                       f_limit=f_limit, h_floor=h_floor, r=fields["r"] if use_r else None,
                       vol=fields["vol"] if use_vol else None, rate_mode=rate_mode, coulomb_mode=coulomb_mode,
                       nthreads=nthreads or oracle.max_threads(), **kw)


def oracle_step_implicit(oracle, otab, un, fields, dt, nsub=1, h_floor=0.0, use_r=False, use_vol=False, coulomb_mode=None, nthreads=0):
    return oracle.step_implicit(otab, un, fields["rho"], fields["bsq"], fields["theta_e"], fields["theta_i"], dt, nsub=nsub,
                                h_floor=h_floor, r=fields["r"] if use_r else None, vol=fields["vol"] if use_vol else None,
                                coulomb_mode=coulomb_mode, nthreads=nthreads or oracle.max_threads())


def rel_err(a, b):
    """Relative error on the updated energies (Theta' is proportional to u' at fixed rho)."""
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    both_nan = np.isnan(a) & np.isnan(b)
    e = np.abs(a - b) / np.maximum(np.abs(b), 1e-300)
    e[both_nan] = 0.0
    return e


def change_err(new_gpu, new_ref, old, thresh=1e-3):
    """Anti-vacuity: relative error of the change (Theta'-Theta) on cells where it exceeds
    ``thresh`` of Theta.  Returns (max error, number of such cells)."""
    old = np.asarray(old, dtype=np.float64)
    dg, dr = new_gpu - old, new_ref - old
    act = np.abs(dr) > thresh * np.abs(old)
    if not act.any():
        return 0.0, 0
    return float((np.abs(dg - dr)[act] / np.abs(dr[act])).max()), int(act.sum())
