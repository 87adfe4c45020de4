"""Radial luminosity profile (numerator of eq 25): per-shell sums of the luminosity terms, computed
inside the same kernel launch, against partial sums of the oracle's per-cell terms.  fp64 atomics make the last bits
order dependent, so the comparison is relative (fp32 cells: the fp32 partial sums of the kernel; fp64 cells: 1e-10)."""
import numpy as np
import pytest

import common as cm
from paper_2505_08855_b200 import api, synth

pytestmark = pytest.mark.gpu

NR, NTH, NPH = 12, 16, 32            # shell = 512 cells (a multiple of the 128-cell warp tile)
SHELL = NTH * NPH


def _tables(oracle, n, nc):
    desc, data, coul = cm.build_tables(n, nc=nc)
    return api.cool_table_create(desc, data, coul), cm.oracle_table(oracle, desc, data, coul), cm.oracle_units(oracle, desc)


def _compare(got, ref_shell, ref_diag, rtol, split_abs=0.0):
    """split_abs: extra absolute tolerance on the per-process terms, as a fraction of the shell's total (the fp32 kernels
    form the Compton share as a difference of two rates, (eta - 1) Q_syn, which cancels where eta is within ~1e-6 of 1)."""
    sh = got["lum_shell"]
    assert sh.shape == ref_shell.shape
    scale = np.abs(ref_shell).max(axis=0)
    assert np.all(np.abs(sh - ref_shell) <= rtol * np.abs(ref_shell) + 1e-3 * rtol * scale + split_abs * ref_shell[:, :1])
    assert (ref_shell[:, 0] > 0).sum() >= ref_shell.shape[0] - 1         # a real profile, not zeros
    for k, name in enumerate(("lum_total", "lum_brems", "lum_synch", "lum_compton")):
        assert sh[:, k].sum() == pytest.approx(got["diag"][name], rel=10 * rtol, abs=1e-300)
        assert got["diag"][name] == pytest.approx(ref_diag[name], rel=10 * rtol, abs=1e-300)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n,nc,nsub", [([32, 32, 32], [32, 32], 1), ([64, 64, 64], [64, 64], 2), ([12, 10, 14, 11], [24, 20], 4)])
def test_shell_sums_explicit(oracle, dtype, n, nc, nsub):
    table, otab, un = _tables(oracle, n, nc)
    f = synth.mad_like_cells(NR, NTH, NPH, dtype=dtype, config=3)
    dt = 50.0
    o = oracle.step(otab, un, f["rho"], f["bsq"], f["theta_e"], f["theta_i"], dt, nsub=nsub, vol=f["vol"], want_cell_lum=True,
                    nthreads=oracle.max_threads())
    ref = oracle.shell_sums(o["cell_lum"], SHELL)
    variants = [api.COOL_V_GLOBAL, api.COOL_V_TEX_POINT] + ([api.COOL_V_SMEM] if n[0] == 32 else [])
    for v in variants:
        got = cm.gpu_step(table, f, dtype, dt, nsub=nsub, variant=v, use_vol=True, shell_cells=SHELL)
        _compare(got, ref, o["diag"], 3e-6 if dtype == np.float32 else 1e-10)
        if len(n) == 3:
            assert np.all(got["lum_shell"][:, 1:] == 0.0)              # no per-process split without process tables
    # ragged: the last shell is partial, the arrays are misaligned (scalar path)
    m = 5 * SHELL + 384
    g = {k: v[:m] for k, v in f.items()}
    og = oracle.step(otab, un, g["rho"], g["bsq"], g["theta_e"], g["theta_i"], dt, nsub=nsub, vol=g["vol"], want_cell_lum=True)
    got = cm.gpu_step(table, g, dtype, dt, nsub=nsub, use_vol=True, shell_cells=SHELL, offset=1, variant=api.COOL_V_GLOBAL)
    _compare(got, oracle.shell_sums(og["cell_lum"], SHELL), og["diag"], 3e-6 if dtype == np.float32 else 1e-10)
    table.destroy()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_shell_sums_implicit_and_analytic(oracle, dtype):
    table, otab, un = _tables(oracle, [12, 10, 14, 11], [24, 20])
    f = synth.mad_like_cells(NR, NTH, NPH, dtype=dtype, config=3)
    dt = 200.0
    o = oracle.step_implicit(otab, un, f["rho"], f["bsq"], f["theta_e"], f["theta_i"], dt, nsub=2, vol=f["vol"], want_cell_lum=True,
                             nthreads=oracle.max_threads())
    got = cm.gpu_step(table, f, dtype, dt, nsub=2, use_vol=True, shell_cells=SHELL, scheme=api.COOL_SCHEME_IMPLICIT)
    _compare(got, oracle.shell_sums(o["cell_lum"], SHELL), o["diag"], 2e-5 if dtype == np.float32 else 1e-9,
             split_abs=1e-6 if dtype == np.float32 else 0.0)
    # analytic variant: shells add up to its own total
    got = cm.gpu_step(table, f, dtype, 1.0, use_vol=True, shell_cells=SHELL, variant=api.COOL_V_ANALYTIC)
    assert got["lum_shell"][:, 0].sum() == pytest.approx(got["diag"]["lum_total"], rel=1e-9)
    table.destroy()


def test_shell_sums_host_path_and_errors(oracle):
    import torch
    table, otab, un = _tables(oracle, [32, 32, 32], [32, 32])
    f = synth.mad_like_cells(NR, NTH, NPH, dtype=np.float32, config=3)
    n = f["rho"].size
    o = oracle.step(otab, un, f["rho"], f["bsq"], f["theta_e"], f["theta_i"], 50.0, vol=f["vol"], want_cell_lum=True)
    ref = oracle.shell_sums(o["cell_lum"], SHELL)
    h = {k: torch.from_numpy(np.ascontiguousarray(f[k])).pin_memory() for k in ("rho", "bsq", "theta_e", "theta_i", "vol")}
    oe, oi = torch.empty(n).pin_memory(), torch.empty(n).pin_memory()
    sh = torch.full((4 * NR,), -1.0, dtype=torch.float64).pin_memory()
    p = api.make_params(50.0)
    d = api.cool_apply_host(table, n, api.COOL_F32, h["rho"], h["bsq"], h["theta_e"], h["theta_i"], oe, oi, p, vol=h["vol"],
                            want_diag=True, shell_cells=SHELL, lum_shell=sh)
    _compare(dict(lum_shell=sh.numpy().reshape(-1, 4), diag=d), ref, o["diag"], 3e-6)
    with pytest.raises(api.CoolError) as e1:                           # not a multiple of the warp tile
        cm.gpu_step(table, f, np.float32, 1.0, use_vol=True, shell_cells=100)
    assert e1.value.status == api.COOL_EINVAL
    with pytest.raises(api.CoolError) as e2:                           # needs the diagnostics
        cm.gpu_step(table, f, np.float32, 1.0, use_vol=True, shell_cells=SHELL, want_diag=False)
    assert e2.value.status == api.COOL_EINVAL
    table.destroy()
