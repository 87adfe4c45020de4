"""Thin Python binding of include/cool.h (argument marshalling only; all compute is in the
CUDA kernels of libcool_b200.so).  Same names as the C ABI:

    cool_table_build_host, cool_table_create, cool_apply, cool_apply_host, cool_table_destroy

Arrays are passed as anything with ``data_ptr()`` (torch tensors, device or pinned host),
numpy arrays (host) or plain integer addresses.  The library is loaded on first use and the
import fails loudly when it is missing: there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcool_b200.so")

COOL_OK, COOL_EINVAL, COOL_ENOMEM, COOL_ECUDA, COOL_EUNSUPPORTED = range(5)
COOL_F32, COOL_F64 = 0, 1
COOL_AX_LOG_RHO, COOL_AX_LOG_THETA_E, COOL_AX_LOG_BSQ, COOL_AX_LOG_THETA_I = range(4)
COOL_AX_LOG_HTH, COOL_AX_LOG_B, COOL_AX_LOG_NE, COOL_AX_LOG_TE = range(4, 8)          # the paper's table (cgs units)
COOL_V_AUTO, COOL_V_TEX_POINT, COOL_V_TEX_HWFILTER, COOL_V_SMEM, COOL_V_GLOBAL, COOL_V_ANALYTIC = range(6)
COOL_COULOMB_AUTO, COOL_COULOMB_OFF, COOL_COULOMB_TABLE, COOL_COULOMB_ANALYTIC = range(4)
COOL_SCHEME_EXPLICIT, COOL_SCHEME_IMPLICIT = range(2)
VARIANT_NAMES = {COOL_V_AUTO: "auto", COOL_V_TEX_POINT: "tex_point", COOL_V_TEX_HWFILTER: "tex_hwfilter",
                 COOL_V_SMEM: "smem", COOL_V_GLOBAL: "global", COOL_V_ANALYTIC: "analytic"}
VARIANTS = {v: k for k, v in VARIANT_NAMES.items()}


class CoolError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"cool status {status}: {msg}")
        self.status = status


class cool_units(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("rho_scale_cgs", "mbh_msun", "gamma_e", "gamma_i", "ln_lambda",
                                          "ion_theta_mass_ratio", "hth_cm", "r_ref_rg", "spin")]


class cool_table_desc(C.Structure):
    _fields_ = [("ndim", C.c_int), ("axis", C.c_int * 4), ("n", C.c_int * 4),
                ("lo", C.c_double * 4), ("hi", C.c_double * 4), ("nproc", C.c_int),
                ("host_data", C.c_void_p * 3), ("host_coulomb", C.c_void_p),
                ("nc", C.c_int * 2), ("clo", C.c_double * 2), ("chi", C.c_double * 2),
                ("units", cool_units),
                ("host_coulomb3", C.c_void_p), ("nc3", C.c_int * 3), ("c3lo", C.c_double * 3), ("c3hi", C.c_double * 3)]


class cool_cells(C.Structure):
    _fields_ = [("ncell", C.c_longlong), ("dtype", C.c_int),
                ("rho", C.c_void_p), ("bsq", C.c_void_p),
                ("theta_e_in", C.c_void_p), ("theta_i_in", C.c_void_p),
                ("theta_e_out", C.c_void_p), ("theta_i_out", C.c_void_p),
                ("r", C.c_void_p), ("vol", C.c_void_p), ("shell_cells", C.c_longlong), ("lum_shell", C.c_void_p),
                ("flags", C.c_void_p)]


class cool_params(C.Structure):
    _fields_ = [("dt", C.c_double), ("nsub", C.c_int), ("f_limit", C.c_double), ("h_floor", C.c_double),
                ("variant", C.c_int), ("coulomb", C.c_int), ("scheme", C.c_int)]


class cool_diag(C.Structure):
    _fields_ = [("lum_total", C.c_double), ("lum_brems", C.c_double), ("lum_synch", C.c_double),
                ("lum_compton", C.c_double), ("n_limited", C.c_longlong), ("n_floored", C.c_longlong),
                ("n_clamped", C.c_longlong)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


DIAG_BYTES = C.sizeof(cool_diag)
EXPORTS = ("cool_table_build_host", "cool_table_create", "cool_apply", "cool_apply_host",
           "cool_table_auto_variant", "cool_last_launch_count", "cool_table_destroy",
           "cool_last_error", "cool_version", "cool_radpress_correct", "cool_last_kernel_name", "cool_table_build_device",
           "cool_apply_noalloc")

_lib = None


def lib():
    """Load libcool_b200.so (built in-tree by ``python -m paper_2505_08855_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2505_08855_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.cool_table_build_host.restype = C.c_int
        L.cool_table_build_host.argtypes = [C.POINTER(cool_table_desc), C.POINTER(C.c_void_p), C.c_void_p, C.c_int]
        L.cool_table_build_device.restype = C.c_int
        L.cool_table_build_device.argtypes = [C.POINTER(cool_table_desc), C.c_int, C.c_void_p]
        L.cool_table_create.restype = C.c_int
        L.cool_table_create.argtypes = [C.POINTER(cool_table_desc), C.c_int, C.POINTER(C.c_void_p)]
        L.cool_apply.restype = C.c_int
        L.cool_apply.argtypes = [C.c_void_p, C.POINTER(cool_cells), C.POINTER(cool_params), C.c_void_p, C.c_void_p]
        L.cool_apply_noalloc.restype = C.c_int
        L.cool_apply_noalloc.argtypes = [C.c_void_p, C.POINTER(cool_cells), C.POINTER(cool_params), C.c_void_p, C.c_void_p]
        L.cool_apply_host.restype = C.c_int
        L.cool_apply_host.argtypes = [C.c_void_p, C.POINTER(cool_cells), C.POINTER(cool_params), C.POINTER(cool_diag)]
        L.cool_table_auto_variant.restype = C.c_int
        L.cool_table_auto_variant.argtypes = [C.c_void_p]
        L.cool_last_launch_count.restype = C.c_int
        L.cool_last_kernel_name.restype = C.c_char_p
        L.cool_table_destroy.restype = C.c_int
        L.cool_table_destroy.argtypes = [C.c_void_p]
        L.cool_radpress_correct.restype = C.c_int
        L.cool_radpress_correct.argtypes = [C.POINTER(cool_units), C.c_longlong, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                            C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.cool_last_error.restype = C.c_char_p
        L.cool_version.restype = C.c_char_p
        _lib = L
    return _lib


def _check(status):
    if status != COOL_OK:
        raise CoolError(status, lib().cool_last_error().decode())


def _ptr(a):
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if hasattr(a, "data_ptr"):
        return a.data_ptr()
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    raise TypeError(f"cannot take the address of {type(a)}")


def default_units(**kw) -> cool_units:
    """Defaults of DESIGN.md: EXP_HIGH rho_scale, M = 10 Msun (L220),
    gamma = 5/3 and a = 0.9375 (L207), ln Lambda = 20 (L147), H_th = 10 r_g, r_ref = 10 r_g."""
    d = dict(rho_scale_cgs=3e-7, mbh_msun=10.0, gamma_e=5.0 / 3.0, gamma_i=5.0 / 3.0, ln_lambda=20.0,
             ion_theta_mass_ratio=1.0, hth_cm=1.476625e7, r_ref_rg=10.0, spin=0.9375)
    d.update(kw)
    return cool_units(**d)


def make_desc(axis, n, lo, hi, nproc, units=None, nc=None, clo=None, chi=None, nc3=None, c3lo=None, c3hi=None) -> cool_table_desc:
    d = cool_table_desc()
    d.ndim = len(n)
    for k in range(d.ndim):
        d.axis[k] = int(axis[k]); d.n[k] = int(n[k]); d.lo[k] = float(lo[k]); d.hi[k] = float(hi[k])
    d.nproc = int(nproc)
    if nc is not None:
        d.nc[0], d.nc[1] = int(nc[0]), int(nc[1])
        d.clo[0], d.clo[1] = float(clo[0]), float(clo[1])
        d.chi[0], d.chi[1] = float(chi[0]), float(chi[1])
    if nc3 is not None:
        for k in range(3):
            d.nc3[k] = int(nc3[k]); d.c3lo[k] = float(c3lo[k]); d.c3hi[k] = float(c3hi[k])
    d.units = units if units is not None else default_units()
    return d


def is_cgs(desc: cool_table_desc) -> bool:
    """The paper's table: axes (log H_th, log B, log n_e, log T_e)."""
    return desc.ndim == 4 and desc.axis[0] == COOL_AX_LOG_HTH


def cool_table_build_host(desc: cool_table_desc, want_coulomb: bool = False, nthreads: int = 0):
    """Host table builder.  Returns (list of nproc float32 arrays of shape n, coulomb array or None)."""
    shape = [desc.n[k] for k in range(desc.ndim)]
    data = [np.empty(shape, dtype=np.float32) for _ in range(desc.nproc)]
    outs = (C.c_void_p * 3)(*[d.ctypes.data for d in data] + [None] * (3 - len(data)))
    if want_coulomb and is_cgs(desc):
        coul = np.empty((desc.nc3[0], desc.nc3[1], desc.nc3[2]), dtype=np.float32)
    else:
        coul = np.empty((desc.nc[0], desc.nc[1]), dtype=np.float32) if want_coulomb else None
    _check(lib().cool_table_build_host(C.byref(desc), outs, None if coul is None else coul.ctypes.data, nthreads))
    return data, coul


def cool_table_build_device(desc: cool_table_desc, device: int = 0):
    """The paper's table tabulated on the GPU (see include/cool.h).  Returns [float32 array of shape n]."""
    out = np.empty([desc.n[k] for k in range(desc.ndim)], dtype=np.float32)
    _check(lib().cool_table_build_device(C.byref(desc), device, out.ctypes.data))
    return [out]


class CoolTable:
    """Owner of an opaque ``cool_table*``."""

    def __init__(self, handle, desc):
        self.handle = handle
        self.desc = desc

    def auto_variant(self) -> int:
        return lib().cool_table_auto_variant(self.handle)

    def destroy(self):
        if self.handle:
            _check(lib().cool_table_destroy(self.handle))
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def cool_table_create(desc: cool_table_desc, data, coulomb=None, device: int = 0) -> CoolTable:
    """Upload a table (list of nproc float32 host arrays, optional Coulomb coefficient array)."""
    keep = [np.ascontiguousarray(d, dtype=np.float32) for d in data]
    if len(keep) != desc.nproc:
        raise ValueError("len(data) != desc.nproc")
    for p in range(3):
        desc.host_data[p] = keep[p].ctypes.data if p < len(keep) else None
    ck = None
    desc.host_coulomb = None
    desc.host_coulomb3 = None
    if coulomb is not None:
        ck = np.ascontiguousarray(coulomb, dtype=np.float32)
        if is_cgs(desc):
            if ck.shape != (desc.nc3[0], desc.nc3[1], desc.nc3[2]):
                raise ValueError("coulomb shape != desc.nc3")
            desc.host_coulomb3 = ck.ctypes.data
        else:
            if ck.shape != (desc.nc[0], desc.nc[1]):
                raise ValueError("coulomb shape != desc.nc")
            desc.host_coulomb = ck.ctypes.data
    h = C.c_void_p()
    _check(lib().cool_table_create(C.byref(desc), device, C.byref(h)))
    for p in range(3):
        desc.host_data[p] = None
    desc.host_coulomb = None
    desc.host_coulomb3 = None
    return CoolTable(h, desc)


def _cells(ncell, dtype, rho, bsq, theta_e_in, theta_i_in, theta_e_out, theta_i_out, r, vol, shell_cells=0, lum_shell=None, flags=None):
    c = cool_cells()
    c.shell_cells = int(shell_cells); c.lum_shell = _ptr(lum_shell); c.flags = _ptr(flags)
    c.ncell = int(ncell); c.dtype = int(dtype)
    c.rho, c.bsq = _ptr(rho), _ptr(bsq)
    c.theta_e_in, c.theta_i_in = _ptr(theta_e_in), _ptr(theta_i_in)
    c.theta_e_out, c.theta_i_out = _ptr(theta_e_out), _ptr(theta_i_out)
    c.r, c.vol = _ptr(r), _ptr(vol)
    return c


def make_params(dt, nsub=1, f_limit=0.3, h_floor=0.0, variant=COOL_V_AUTO, coulomb=COOL_COULOMB_AUTO,
                scheme=COOL_SCHEME_EXPLICIT) -> cool_params:
    return cool_params(float(dt), int(nsub), float(f_limit), float(h_floor), int(variant), int(coulomb), int(scheme))


def cool_apply(table: CoolTable, ncell, dtype, rho, bsq, theta_e_in, theta_i_in, theta_e_out, theta_i_out,
               params: cool_params, r=None, vol=None, d_diag=None, stream=None, shell_cells=0, lum_shell=None, flags=None):
    """Asynchronous update of DEVICE arrays on ``stream`` (a cudaStream_t address; None = default).
    ``lum_shell``: optional device float64 array of 4*ceil(ncell/shell_cells) (radial luminosity profile);
    ``flags``: optional device uint8 array of ncell per-cell event flags (see include/cool.h)."""
    c = _cells(ncell, dtype, rho, bsq, theta_e_in, theta_i_in, theta_e_out, theta_i_out, r, vol, shell_cells, lum_shell, flags)
    _check(lib().cool_apply(table.handle, C.byref(c), C.byref(params), _ptr(d_diag), stream))


COOL_NOALLOC_MAX_CELLS = 1 << 24
COOL_NOALLOC_SCRATCH_BYTES = 4 << 20


def cool_apply_noalloc(table: CoolTable, ncell, dtype, rho, bsq, theta_e_in, theta_i_in, theta_e_out, theta_i_out,
                       params: cool_params, r=None, vol=None, d_diag=None, stream=None, flags=None):
    """``cool_apply`` with the step's scratch in a static device array: no allocation inside the call (include/cool.h).
    At most COOL_NOALLOC_MAX_CELLS cells, no radial profile; calls that overlap on the GPU race on the shared scratch."""
    c = _cells(ncell, dtype, rho, bsq, theta_e_in, theta_i_in, theta_e_out, theta_i_out, r, vol, 0, None, flags)
    _check(lib().cool_apply_noalloc(table.handle, C.byref(c), C.byref(params), _ptr(d_diag), stream))


def cool_apply_host(table: CoolTable, ncell, dtype, rho, bsq, theta_e_in, theta_i_in, theta_e_out, theta_i_out,
                    params: cool_params, r=None, vol=None, want_diag=False, shell_cells=0, lum_shell=None, flags=None):
    """Synchronous update of HOST arrays (copies staged and overlapped inside the library).
    ``lum_shell``: optional host float64 array of 4*ceil(ncell/shell_cells) (radial luminosity profile);
    ``flags``: optional host uint8 array of ncell per-cell event flags."""
    c = _cells(ncell, dtype, rho, bsq, theta_e_in, theta_i_in, theta_e_out, theta_i_out, r, vol, shell_cells, lum_shell, flags)
    d = cool_diag() if want_diag else None
    _check(lib().cool_apply_host(table.handle, C.byref(c), C.byref(params), None if d is None else C.byref(d)))
    return None if d is None else d.as_dict()


def cool_radpress_correct(units: cool_units, ncell, dtype, rho, theta_e, hscale, tau_crit, theta_e_out, d_ncorrected=None, stream=None):
    """Radiation-pressure temperature correction (eq 29) of DEVICE arrays on the current device; see include/cool.h."""
    _check(lib().cool_radpress_correct(C.byref(units), int(ncell), int(dtype), _ptr(rho), _ptr(theta_e), _ptr(hscale),
                                       float(tau_crit), _ptr(theta_e_out), _ptr(d_ncorrected), stream))


def cool_table_destroy(table: CoolTable):
    table.destroy()


def cool_last_launch_count() -> int:
    return lib().cool_last_launch_count()


def cool_last_kernel_name() -> str:
    return lib().cool_last_kernel_name().decode()


def cool_version() -> str:
    return lib().cool_version().decode()
