"""Seeded synthetic cell fields.

This module serves BOTH the oracle-side tests and the CUDA path.  It holds none of the
method's arithmetic: only shapes, ranges and random draws.  It stands in for H-AMR
snapshots (Table I), which do not exist outside the
authors' runs.  numpy only; importing it never touches CUDA.

Streams are counter-based (Philox keyed by (MASTER_SEED, config, field)), so any field of
any config can be regenerated independently and in any order.
"""
from __future__ import annotations

import numpy as np

MASTER_SEED = 20250508

# log10 ranges of the BASELINE.json configs (also the table ranges)
LOG_RHO = (-6.0, 0.0)
LOG_THETA = (-3.0, 1.5)
LOG_BSQ = (-8.0, 0.0)

_F_RHO, _F_THE, _F_THI, _F_BSQ, _F_OUT_SEL, _F_OUT_AX, _F_OUT_VAL, _F_BETA, _F_NOISE = range(9)


def _rng(config: int, field: int, seed: int = MASTER_SEED) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), (int(config) << 8) | int(field)]))


def _uniform(config, field, n, lo, hi, seed):
    return _rng(config, field, seed).uniform(lo, hi, size=n)


def log_uniform_cells(ncell: int, dtype=np.float32, config: int = 2, outlier_frac: float = 0.0,
                      seed: int = MASTER_SEED):
    """Configs 1, 2, 4 and the worst-locality form of config 5: independent log-uniform
    rho, Theta_e, Theta_i, bsq on the table ranges.  With ``outlier_frac`` > 0 (config 2:
    0.01) that fraction of cells gets one random coordinate moved outside the range by
    lo - U(0,1) or hi + U(0,1) dex, to exercise clamping.

    Returns dict(rho, theta_e, theta_i, bsq) of 1-D arrays of ``dtype``."""
    lr = _uniform(config, _F_RHO, ncell, *LOG_RHO, seed)
    le = _uniform(config, _F_THE, ncell, *LOG_THETA, seed)
    li = _uniform(config, _F_THI, ncell, *LOG_THETA, seed)
    lb = _uniform(config, _F_BSQ, ncell, *LOG_BSQ, seed)
    if outlier_frac > 0.0:
        sel = _rng(config, _F_OUT_SEL, seed).random(ncell) < outlier_frac
        ax = _rng(config, _F_OUT_AX, seed).integers(0, 8, size=ncell)   # axis*2 + side
        val = _rng(config, _F_OUT_VAL, seed).random(ncell)
        for a, (arr, (lo, hi)) in enumerate(((lr, LOG_RHO), (le, LOG_THETA), (lb, LOG_BSQ), (li, LOG_THETA))):
            low = sel & (ax == 2 * a)
            high = sel & (ax == 2 * a + 1)
            arr[low] = lo - val[low]
            arr[high] = hi + val[high]
    out = dict(rho=10.0 ** lr, theta_e=10.0 ** le, theta_i=10.0 ** li, bsq=10.0 ** lb)
    return {k: v.astype(dtype) for k, v in out.items()}


def mad_like_cells(nr: int = 288, nth: int = 192, nph: int = 144, dtype=np.float32, config: int = 3,
                   smooth_beta: bool = False, r_in: float = 1.2, r_out: float = 1000.0,
                   seed: int = MASTER_SEED):
    """Config 3 (and the coherent form of config 5 when called with 512^3): MAD-like
    torus on an (r, theta, phi) grid, phi fastest, r log-spaced on [r_in, r_out] r_g:

        rho     = (r/r0)^-1.5 exp(-(theta - pi/2)^2 / 0.3^2),   r0 = r_in
        Theta_i = 30 (r/r0)^-1,   Theta_e = 3 (r/r0)^-1
        bsq     = rho / beta,  beta log-uniform in [0.1, 100] per cell
                  (``smooth_beta``: beta = 10^(sin(4 phi) * cos(theta)) varies smoothly)
        every field times exp(0.05 N(0,1))   (5 % log-normal noise)

    Returns dict(rho, theta_e, theta_i, bsq, r, vol, shape); r is the cell radius in r_g
    (for the temperature floor) and vol the flat-space cell volume r^3 sin(theta)
    dlnr dtheta dphi (for the luminosity diagnostic)."""
    n = nr * nth * nph
    lnr = np.linspace(np.log(r_in), np.log(r_out), nr)
    r1 = np.exp(lnr)
    th1 = (np.arange(nth) + 0.5) * np.pi / nth
    ph1 = (np.arange(nph) + 0.5) * 2.0 * np.pi / nph
    R = r1[:, None, None]
    TH = th1[None, :, None]
    PH = ph1[None, None, :]
    x = R / r_in
    rho = np.broadcast_to(x ** -1.5 * np.exp(-((TH - 0.5 * np.pi) ** 2) / 0.3 ** 2), (nr, nth, nph))
    thi = np.broadcast_to(30.0 / x, (nr, nth, nph))
    the = np.broadcast_to(3.0 / x, (nr, nth, nph))
    if smooth_beta:
        beta = 10.0 ** np.broadcast_to(np.sin(4.0 * PH) * np.cos(TH), (nr, nth, nph))
    else:
        beta = 10.0 ** _uniform(config, _F_BETA, n, -1.0, 2.0, seed).reshape(nr, nth, nph)
    bsq = rho / beta
    out = {}
    for k, (name, arr) in enumerate((("rho", rho), ("theta_e", the), ("theta_i", thi), ("bsq", bsq))):
        noise = _rng(config, (_F_NOISE << 4) | k, seed).standard_normal(n, dtype=np.float32)
        out[name] = (arr.reshape(-1) * np.exp(0.05 * noise.astype(np.float64))).astype(dtype)
    dlnr = (lnr[-1] - lnr[0]) / (nr - 1)
    vol = R ** 3 * np.sin(TH) * dlnr * (np.pi / nth) * (2.0 * np.pi / nph)
    out["r"] = np.broadcast_to(R, (nr, nth, nph)).reshape(-1).astype(dtype)
    out["vol"] = np.broadcast_to(vol, (nr, nth, nph)).reshape(-1).astype(dtype)
    out["shape"] = (nr, nth, nph)
    return out


def scale_height(r, r_tr: float = 50.0, thick: float = 0.3, thin: float = 0.05):
    """Density scale height H(r) in r_g of a truncated disc as in the paper's Fig. 4: H/r = ``thick`` inside the
    truncation radius ``r_tr``, falling to ``thin`` outside:  H = r (thin + (thick - thin)/(1 + (r/r_tr)^4))."""
    r = np.asarray(r, dtype=np.float64)
    return r * (thin + (thick - thin) / (1.0 + (r / r_tr) ** 4))


def thick_disc_cells(nr: int = 288, nth: int = 192, nph: int = 144, dtype=np.float32, config: int = 6, rho0: float = 5.0,
                     r_in: float = 1.2, r_out: float = 300.0, seed: int = MASTER_SEED):
    """Input of the radiation-pressure correction (the high-accretion-rate runs after the disc has
    collapsed): an (r, theta, phi) grid as in mad_like_cells with

        rho     = rho0 exp(-(theta - pi/2)^2 / (2 (H/r)^2)),  H(r) = scale_height(r)     (code units of rho_scale)
        Theta_e = 3 (r/r_in)^-1   (T_e ~ 1e9 K near r ~ 20 r_g)
        hscale  = H(r) in r_g, the same for every cell of a radial shell
        rho and Theta_e times exp(0.05 N(0,1))

    With Table I's rho_scale = 3e-7 g/cm^3 and M = 10 Msun this gives tau_sca = n_e sigma_T H of a few in the midplane
    (the paper quotes 2-8, L338) and << 1 off the midplane.  Returns dict(rho, theta_e, r, hscale, shape)."""
    n = nr * nth * nph
    r1 = np.exp(np.linspace(np.log(r_in), np.log(r_out), nr))
    th1 = (np.arange(nth) + 0.5) * np.pi / nth
    R = r1[:, None, None]
    TH = th1[None, :, None]
    H = scale_height(R)
    rho = np.broadcast_to(rho0 * np.exp(-((TH - 0.5 * np.pi) ** 2) / (2.0 * (H / R) ** 2)), (nr, nth, nph))
    the = np.broadcast_to(3.0 * r_in / R, (nr, nth, nph))
    out = {}
    for k, (name, arr) in enumerate((("rho", rho), ("theta_e", the))):
        noise = _rng(config, (_F_NOISE << 4) | k, seed).standard_normal(n, dtype=np.float32)
        out[name] = (arr.reshape(-1) * np.exp(0.05 * noise.astype(np.float64))).astype(dtype)
    out["r"] = np.broadcast_to(R, (nr, nth, nph)).reshape(-1).astype(dtype)
    out["hscale"] = np.broadcast_to(H, (nr, nth, nph)).reshape(-1).astype(dtype)
    out["shape"] = (nr, nth, nph)
    return out


# rho_scale [g cm^-3] for the density-normalisation sweep of config 3: log-log
# interpolation of (mdot, rho_scale) through PAPER.md Table I (L290-L294):
# (2.6e-1, 3e-7), (5.1e-4, 1e-8), (4.7e-6, 1e-9).
_TABLE_I = ((4.7e-6, 1e-9), (5.1e-4, 1e-8), (2.6e-1, 3e-7))


def rho_scale_for_mdot(mdot: float) -> float:
    lm = np.log10([m for m, _ in _TABLE_I])
    ls = np.log10([s for _, s in _TABLE_I])
    x = np.log10(mdot)
    if x <= lm[1]:
        k = 0
    else:
        k = 1
    slope = (ls[k + 1] - ls[k]) / (lm[k + 1] - lm[k])
    return float(10.0 ** (ls[k] + slope * (x - lm[k])))


def shard_range(ncell: int, rank: int, world: int):
    """Contiguous cell range [lo, hi) owned by ``rank`` of ``world``."""
    base, rem = divmod(int(ncell), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
