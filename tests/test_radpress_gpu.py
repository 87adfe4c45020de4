"""Radiation-pressure temperature correction (eq 29; reading C-20): the CUDA kernel behind
cool_radpress_correct against oracle Part C, element by element.  Bar: 1e-5 (fp32 cells) / 1e-12 (fp64 cells) on the
corrected Theta_e.  The decision tau_sca > tau_crit is taken in the cells' precision by the kernel and in fp64 by the
oracle: cells within 4 ulp of the threshold may go either way, and must then equal one of the two valid answers."""
import numpy as np
import pytest
import torch

import common as cm
from paper_2505_08855_b200 import api, synth

pytestmark = pytest.mark.gpu
TOL = {np.float32: 1e-5, np.float64: 1e-12}


def _gpu(units, rho, the, hs, dtype, tau_crit, offset=0, inplace=False, count=True):
    """offset: element offset of every array inside its allocation (1 = not 16-byte aligned: scalar path)."""
    n = rho.size
    tdt = torch.float32 if dtype == np.float32 else torch.float64
    dev = torch.device("cuda:0")

    def put(a):
        t = torch.empty(n + offset, dtype=tdt, device=dev)
        t[offset:] = torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).to(dev)
        return t[offset:]
    d_rho, d_the, d_hs = put(rho), put(the), put(hs)
    d_out = d_the if inplace else torch.full((n + offset,), -7.0, dtype=tdt, device=dev)[offset:]
    d_cnt = torch.full((1,), -1, dtype=torch.int64, device=dev) if count else None
    api.cool_radpress_correct(units, n, api.COOL_F32 if dtype == np.float32 else api.COOL_F64, d_rho, d_the, d_hs, tau_crit,
                              d_out, d_cnt)
    torch.cuda.synchronize()
    assert api.cool_last_launch_count() == (1 if n else 0)
    return d_out.cpu().numpy().astype(np.float64), (int(d_cnt.item()) if count else None)


def _check(oracle, un, rho, the, hs, dtype, tau_crit, got, cnt):
    """Oracle on the values the kernel saw (the cells rounded to dtype)."""
    rho64, the64, hs64 = (np.asarray(a, dtype=dtype).astype(np.float64) for a in (rho, the, hs))
    ref, _ = oracle.radpress(un, rho64, the64, hs64, tau_crit=tau_crit)
    tau_all = oracle.tau_sca(un, 1.0, 1.0) * rho64 * hs64               # tau_sca is linear in rho and H (L353)
    eps = np.finfo(dtype).eps
    border = np.abs(tau_all - tau_crit) <= 4 * eps * tau_crit
    ok = ~border
    nan = np.isnan(ref)
    assert np.array_equal(np.isnan(got), nan)
    sel = ok & ~nan & (ref != 0)
    assert np.array_equal(got[ok & ~nan & (ref == 0)], ref[ok & ~nan & (ref == 0)])
    err = np.abs(got - ref)[sel] / np.abs(ref[sel])
    assert err.size == 0 or err.max() <= TOL[dtype], err.max()
    if border.any():                                                    # either decision is valid there
        alt, _ = oracle.radpress(un, rho64[border], the64[border], hs64[border], tau_crit=tau_crit * (1 - 1e-3))
        b = got[border]
        assert np.all((np.abs(b - ref[border]) <= TOL[dtype] * np.abs(b)) | (np.abs(b - alt) <= TOL[dtype] * np.abs(b)))
    with np.errstate(invalid="ignore"):
        thick = (tau_all > tau_crit) & (rho64 > 0) & (the64 > 0)
    assert np.array_equal(got[~thick & ok & ~nan], the64[~thick & ok & ~nan])   # thin cells are copied bit for bit
    if cnt is not None:
        assert abs(cnt - int(thick.sum())) <= int(border.sum())
    return err.max() if err.size else 0.0, int(thick.sum())


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("tau_crit", [1.0, 4.6])
def test_mad_like_disc(oracle, dtype, tau_crit):
    """The paper's use: a disc with an optically thick outer part (tau_sca of a few, L338); several tiles + a ragged tail."""
    units = api.default_units()
    un = oracle.Units(units.rho_scale_cgs, units.mbh_msun)
    f = synth.thick_disc_cells(40, 48, 37, dtype=dtype)
    n = f["rho"].size - 3                                                # 71037: not a multiple of 4 or of the CTA tile
    rho, the, hs = f["rho"][:n], f["theta_e"][:n], f["hscale"][:n]
    got, cnt = _gpu(units, rho, the, hs, dtype, tau_crit)
    err, nthick = _check(oracle, un, rho, the, hs, dtype, tau_crit, got, cnt)
    assert 0.02 * n < nthick < 0.5 * n                                   # both kinds of cell present
    # unaligned arrays (scalar path), in place, without the counter: same numbers bit for bit
    got2, _ = _gpu(units, rho, the, hs, dtype, tau_crit, offset=1, inplace=True, count=False)
    assert np.array_equal(got2, got, equal_nan=True)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_all_regimes_and_degenerate_cells(oracle, dtype):
    """Log-uniform cells: beta = a T_e^3/(N k) spans ~40 decades, from gas- to radiation-dominated; plus the degenerate cells."""
    units = api.default_units(rho_scale_cgs=1.0)                         # dense: reaches beta << 1
    un = oracle.Units(units.rho_scale_cgs, units.mbh_msun)
    rng = np.random.default_rng(17)
    n = 200_003
    rho = 10 ** rng.uniform(-6, 6, n)
    the = 10 ** rng.uniform(-9, 1.5, n)
    hs = 10 ** rng.uniform(-3, 2, n)
    rho[5] = 0.0; rho[6] = -1.0; the[7] = 0.0; the[8] = -2.0; the[9] = np.nan; rho[10] = np.nan; hs[11] = np.nan
    got, cnt = _gpu(units, rho, the, hs, dtype, 0.0)
    err, nthick = _check(oracle, un, rho, the, hs, dtype, 0.0, got, cnt)
    y = got / np.asarray(the, dtype=dtype).astype(np.float64)
    with np.errstate(invalid="ignore"):
        assert (y < 1e-3).sum() > 1000 and ((y > 0.1) & (y < 0.9)).sum() > 1000 and (y > 0.999999).sum() > 1000
    assert nthick == cnt


def test_empty_and_errors():
    units = api.default_units()
    api.cool_radpress_correct(units, 0, api.COOL_F32, None, None, None, 1.0, None, None)
    assert api.cool_last_launch_count() == 0
    x = torch.ones(8, device="cuda:0")
    with pytest.raises(api.CoolError):
        api.cool_radpress_correct(units, 8, api.COOL_F32, x, x, None, 1.0, x)
    with pytest.raises(api.CoolError):
        api.cool_radpress_correct(units, 8, api.COOL_F32, x, x, x, -1.0, x)
    with pytest.raises(api.CoolError):
        api.cool_radpress_correct(units, -1, api.COOL_F32, x, x, x, 1.0, x)
    with pytest.raises(api.CoolError):
        api.cool_radpress_correct(units, 8, 7, x, x, x, 1.0, x)


def test_fullsize_sampled(oracle):
    """512^3 fp32 cells in the launch configuration bench.py times; 200 000 sampled cells against the oracle, and the
    properties that hold at any size (0 < out <= in, thin cells untouched, counter = thick cells)."""
    units = api.default_units()
    un = oracle.Units(units.rho_scale_cgs, units.mbh_msun)
    f = synth.thick_disc_cells(512, 512, 512)
    hs = f["hscale"]
    dev = torch.device("cuda:0")
    d_rho, d_the, d_hs = (torch.from_numpy(a).to(dev) for a in (f["rho"], f["theta_e"], hs))
    d_out = torch.empty_like(d_the)
    d_cnt = torch.zeros(1, dtype=torch.int64, device=dev)
    api.cool_radpress_correct(units, d_rho.numel(), api.COOL_F32, d_rho, d_the, d_hs, 1.0, d_out, d_cnt)
    torch.cuda.synchronize()
    assert bool(((d_out >= 0) & (d_out <= d_the)).all())      # rho underflows to 0 far off the midplane
    changed = int((d_out != d_the).sum().item())
    assert changed == int(d_cnt.item()) and 0 < changed < d_rho.numel()
    idx = np.random.default_rng(5).choice(d_rho.numel(), 200_000, replace=False)
    idx.sort()
    got = d_out.cpu().numpy()[idx].astype(np.float64)
    _check(oracle, un, f["rho"][idx], f["theta_e"][idx], hs[idx], np.float32, 1.0, got, None)
