"""Parity of the implicit scheme (COOL_SCHEME_IMPLICIT; PAPER.md L185 (ii), reading C-18) through the C ABI against
oracle Part B'.  The CUDA path finds the root by a node search plus safeguarded false position, the oracle by plain
bisection.  fp64 cells: fp64 solve, both stop within an ulp or two of the root (1e-10).  fp32 cells: the fp32 solve on the T'
tables locates the root, an fp64 secant-Newton step in the interval coordinate refines it, and the state between sub-steps
is carried in fp64: north_star's 1e-5.
Where Lambda is not monotone in Theta_e several roots can exist and any of them solves the scheme (reading C-17): EVERY cell
that differs from the oracle is followed sub-step by sub-step (a chain of single-sub-step launches) and each link must
satisfy the oracle's residual; such cells must be rare."""
import numpy as np
import pytest

import common as cm
from paper_2505_08855_b200 import api, synth

pytestmark = pytest.mark.gpu

TOL = {np.float32: 1e-5, np.float64: 1e-10}
IMP = api.COOL_SCHEME_IMPLICIT


def _table(oracle, n, nc):
    desc, data, coul = cm.build_tables(n, nc=nc)
    return api.cool_table_create(desc, data, coul), cm.oracle_table(oracle, desc, data, coul), cm.oracle_units(oracle, desc)


def _check(oracle, otab, un, f, got, ref, dtype, dt, nsub, label, table=None, **kw):
    tol = TOL[dtype]
    ee = cm.rel_err(got["theta_e"], ref["theta_e"]); ei = cm.rel_err(got["theta_i"], ref["theta_i"])
    bad = np.flatnonzero((ee > tol) | (ei > tol))
    assert bad.size <= max(2, int(2e-4 * ee.size)), f"{label}: {bad.size} cells differ, max {ee.max():.2e} {ei.max():.2e}"
    if bad.size:
        # another root of the same equation is a valid answer.  Follow every such cell through its sub-steps with single-
        # sub-step launches (h = dt/nsub): at each link the oracle's F must change sign within tw of the returned Theta_e',
        # and the chain must end where the nsub launch ended.
        assert table is not None
        tw = 5e-6 if dtype == np.float32 else 1e-11
        g = {k: np.ascontiguousarray(v[bad]) for k, v in f.items() if isinstance(v, np.ndarray) and v.shape == f["rho"].shape}
        h = dt / nsub
        for _ in range(nsub):
            one = cm.gpu_step(table, g, dtype, h, nsub=1, scheme=IMP, **kw)
            for j in range(bad.size):
                res = lambda th: oracle.implicit_residual(otab, un, g["rho"][j], g["bsq"][j], g["theta_e"][j], g["theta_i"][j], h, th,
                                                          h_floor=kw.get("h_floor", 0.0), r=g["r"][j] if kw.get("use_r") else 0.0)
                t = one["theta_e"][j]
                # a root: F changes sign within tw of it — or, where F is flat (Lambda/u_e falling like 1/Theta_e in a strongly
                # cooled cell: F' << R/theta, an ill-conditioned root), F vanishes to the rounding of its own terms, which are
                # at least Theta_e in size (backward error)
                ok = res(t * (1 - tw)) <= 0.0 <= res(t * (1 + tw)) or abs(res(t)) <= 0.4 * tw * float(g["theta_e"][j])
                assert ok, (label, int(bad[j]), t, res(t))
            g["theta_e"], g["theta_i"] = one["theta_e"].astype(dtype), one["theta_i"].astype(dtype)
        assert cm.rel_err(g["theta_e"], got["theta_e"][bad]).max() <= 10 * tol, label
        assert cm.rel_err(g["theta_i"], got["theta_i"][bad]).max() <= 10 * tol, label
    assert (got["theta_e"] > 0).all() and (got["theta_i"] > 0).all()
    return max(np.delete(ee, bad).max(), np.delete(ei, bad).max()), bad.size


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("dt,nsub", [(1e-3, 1), (10.0, 1), (1e4, 4)])
def test_implicit_config1_variants(oracle, dtype, dt, nsub):
    """configs[0] shape: 32^3 (+3) log-uniform cells with 1 % outliers, table 64^3, Coulomb 64^2."""
    table, otab, un = _table(oracle, [64, 64, 64], [64, 64])
    f = synth.log_uniform_cells(32 ** 3 + 3, dtype=dtype, config=1, outlier_frac=0.01)
    ref = cm.oracle_step_implicit(oracle, otab, un, f, dt, nsub=nsub)
    base = None
    for v in (api.COOL_V_GLOBAL, api.COOL_V_TEX_POINT, api.COOL_V_AUTO):
        got = cm.gpu_step(table, f, dtype, dt, nsub=nsub, variant=v, scheme=IMP)
        err, nbad = _check(oracle, otab, un, f, got, ref, dtype, dt, nsub, api.VARIANT_NAMES[v], table=table, variant=v)
        print(f"\nimplicit {np.dtype(dtype).name} dt={dt} nsub={nsub} {api.VARIANT_NAMES[v]}: max rel err {err:.2e}, {nbad} cells on another root")
        d, r = got["diag"], ref["diag"]
        assert d["lum_total"] == pytest.approx(r["lum_total"], rel=(2e-6 if nbad == 0 else 2e-5) if dtype == np.float32 else 1e-9)   # a cell on another root moves the sum too
        assert d["n_limited"] == 0 and d["n_clamped"] == r["n_clamped"]
        assert got["launches"] == 1
        if base is None:
            base = got
        else:
            assert np.array_equal(base["theta_e"], got["theta_e"]) and np.array_equal(base["theta_i"], got["theta_i"])
    # anti-vacuity: the step changes many cells, and for large dt it differs from the explicit (limited) scheme
    changed = np.abs(ref["theta_e"] - f["theta_e"]) > 1e-3 * f["theta_e"]
    assert changed.sum() > (300 if dt < 1 else 5000)
    if dt >= 10.0:
        exp = cm.gpu_step(table, f, dtype, dt, nsub=nsub, variant=api.COOL_V_GLOBAL)
        assert (np.abs(exp["theta_e"] - got["theta_e"]) > 1e-2 * got["theta_e"]).sum() > 1000
    for v in (api.COOL_V_TEX_HWFILTER, api.COOL_V_ANALYTIC):
        with pytest.raises(api.CoolError) as ei_:
            cm.gpu_step(table, f, dtype, dt, nsub=nsub, variant=v, scheme=IMP)
        assert ei_.value.status == api.COOL_EUNSUPPORTED
    table.destroy()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_implicit_smem_table_ragged_inplace(oracle, dtype):
    table, otab, un = _table(oracle, [32, 32, 32], [32, 32])
    assert table.auto_variant() == api.COOL_V_SMEM
    f = synth.log_uniform_cells(50001, dtype=dtype, config=2, outlier_frac=0.01)
    ref = cm.oracle_step_implicit(oracle, otab, un, f, 300.0, nsub=2)
    for kw in (dict(variant=api.COOL_V_SMEM), dict(variant=api.COOL_V_GLOBAL, inplace=True), dict(variant=api.COOL_V_AUTO, offset=1)):
        got = cm.gpu_step(table, f, dtype, 300.0, nsub=2, scheme=IMP, **kw)
        _check(oracle, otab, un, f, got, ref, dtype, 300.0, 2, str(kw), table=table)
    # empty input, rho <= 0 and NaN cells
    g = {k: v[:7].copy() for k, v in f.items()}
    g["rho"][1] = 0.0; g["theta_i"][3] = np.nan
    got = cm.gpu_step(table, g, dtype, 300.0, nsub=2, scheme=IMP)
    assert got["theta_e"][1] == g["theta_e"][1] and got["theta_i"][1] == g["theta_i"][1]
    assert np.isnan(got["theta_e"][3]) and np.isnan(got["theta_i"][3]) and np.isfinite(np.delete(got["theta_e"], 3)).all()
    e = {k: v[:0] for k, v in f.items()}
    assert cm.gpu_step(table, e, dtype, 1.0, scheme=IMP)["diag"]["lum_total"] == 0.0
    table.destroy()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_implicit_process_tables_mad_field_floor(oracle, dtype):
    """4-D process tables (eqs 10-14 inside the root solve), MAD-like field, floor, volume weights, luminosity split."""
    table, otab, un = _table(oracle, [12, 10, 14, 11], [24, 20])
    f = synth.mad_like_cells(40, 24, 32, dtype=dtype, config=3)
    for dt, nsub in ((1.0, 1), (1e3, 3)):
        ref = cm.oracle_step_implicit(oracle, otab, un, f, dt, nsub=nsub, h_floor=0.12, use_r=True, use_vol=True)
        got = cm.gpu_step(table, f, dtype, dt, nsub=nsub, h_floor=0.12, use_r=True, use_vol=True, scheme=IMP, variant=api.COOL_V_GLOBAL)
        _check(oracle, otab, un, f, got, ref, dtype, dt, nsub, f"mad dt={dt}", table=table, h_floor=0.12, use_r=True, variant=api.COOL_V_GLOBAL)
        rt = 2e-5 if dtype == np.float32 else 1e-9
        for k in ("lum_total", "lum_brems", "lum_synch", "lum_compton"):
            assert got["diag"][k] == pytest.approx(ref["diag"][k], rel=rt, abs=1e-300), k
        assert 0 < got["diag"]["n_floored"] == ref["diag"]["n_floored"] < f["rho"].size     # h_floor = 0.12 floors part of this field
    table.destroy()
