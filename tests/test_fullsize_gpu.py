"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (same workload recipes, same tables,
same cool_apply call): EVERY cell against the oracle (the oracle does 134 M cells of configs[4] in ~14 s on the box's 16
cores), the luminosity sums and event counts against the oracle's, and anti-vacuity checks (the update must really change
many cells, and the error of the change itself is bounded)."""
import numpy as np
import pytest

import bench
import common as cm
from paper_2505_08855_b200 import api, synth

pytestmark = pytest.mark.gpu

MR = 9.1093837015e-28 / 1.67262192369e-24
CHUNK = 1 << 24                      # cells per oracle call (keeps the fp64 copies of the fields below ~2 GB)


def _oracle_all(oracle, otab, un, f, spec, dt, implicit, keys):
    """The oracle over the whole field, in chunks.  Returns theta_e, theta_i (float64), the summed diagnostics and, for the
    explicit scheme, h Lambda/u_e of the first sub-step (limiter threshold check)."""
    n = f["rho"].size
    the, thi = np.empty(n), np.empty(n)
    ratio = None if implicit else np.empty(n)
    diag = dict(lum_total=0.0, lum_brems=0.0, lum_synch=0.0, lum_compton=0.0, n_limited=0, n_floored=0, n_clamped=0)
    for lo in range(0, n, CHUNK):
        sl = slice(lo, min(lo + CHUNK, n))
        sub = {k: f[k][sl] for k in keys}
        kw = dict(h_floor=spec.get("floor", 0.0), use_r=bool(spec.get("floor")), use_vol=bool(spec.get("vol")))
        if implicit:
            o = cm.oracle_step_implicit(oracle, otab, un, sub, dt, nsub=spec["nsub"], **kw)
        else:
            o = cm.oracle_step(oracle, otab, un, sub, dt, nsub=spec["nsub"], want_rates=True, **kw)
            ratio[sl] = o["lam0"] * (dt / spec["nsub"]) / (sub["rho"].astype(np.float64) * sub["theta_e"].astype(np.float64) * MR * 1.5)
        the[sl], thi[sl] = o["theta_e"], o["theta_i"]
        for k in diag:
            diag[k] += o["diag"][k]
    return the, thi, diag, ratio


def _run_workload(oracle, name, variants, implicit=False, dt=None, tables=None, units_kw=None, gate=1e-5, spec_kw=None):
    import torch
    spec = bench.workload_spec(name)
    spec.update(spec_kw or {})
    dt = spec["dt"] if dt is None else dt
    if tables is None:
        axis, lo, hi = bench.table_ranges(spec["n"])
        desc = api.make_desc(axis, spec["n"], lo, hi, 1 if len(spec["n"]) == 3 else 3, nc=spec["nc"], clo=cm.CLO, chi=cm.CHI,
                             units=api.default_units(**(units_kw or {})))
        data, coul = api.cool_table_build_host(desc, want_coulomb=True)
    else:
        desc, data, coul = tables
    table = api.cool_table_create(desc, data, coul)
    otab, un = cm.oracle_table(oracle, desc, data, coul), cm.oracle_units(oracle, desc)
    f = bench.make_fields(spec)
    n = f["rho"].size
    dev = torch.device("cuda:0")
    keys = ["rho", "bsq", "theta_e", "theta_i"] + (["vol"] if spec.get("vol") else []) + (["r"] if spec.get("floor") else [])
    d = {k: torch.from_numpy(f[k]).to(dev) for k in keys}
    oe = torch.empty(n, dtype=torch.float32, device=dev); oi = torch.empty_like(oe)
    dg = torch.zeros(api.DIAG_BYTES, dtype=torch.uint8, device=dev) if spec["diag"] else None
    idx = None
    if implicit:
        # the oracle's implicit solve is a 200-step bisection per sub-step: 2^22 sampled cells instead of all (the explicit
        # scheme, which bench.py's default line times, is compared cell by cell)
        idx = np.sort(np.random.default_rng(11).choice(n, 1 << 22, replace=False))
        fo = {k: f[k][idx] for k in keys}
        rthe, rthi, rdiag, ratio = _oracle_all(oracle, otab, un, fo, spec, dt, implicit, keys)
    else:
        rthe, rthi, rdiag, ratio = _oracle_all(oracle, otab, un, f, spec, dt, implicit, keys)
    the0 = f["theta_e"].astype(np.float64) if idx is None else f["theta_e"][idx].astype(np.float64)
    near_floor = None
    if spec.get("floor") and not implicit and spec["nsub"] == 1:
        r = f["r"].astype(np.float64)
        tfl = 0.5 * np.pi * (spec["floor"] * r / (r ** 1.5 + 0.9375)) ** 2
        near_floor = np.flatnonzero(np.abs((the0 + f["theta_i"].astype(np.float64)) * MR / tfl - 1.0) <= 4 * 1.2e-7)
        assert near_floor.size <= max(8, 1e-5 * n)
        sub = {k: f[k][near_floor] for k in keys}
        alt_floored = cm.oracle_step(oracle, otab, un, sub, dt, nsub=1, h_floor=1e3, use_r=True, use_vol=bool(spec.get("vol")))
        alt_cooled = cm.oracle_step(oracle, otab, un, sub, dt, nsub=1, h_floor=0.0, use_r=True, use_vol=bool(spec.get("vol")))
        print(f"\n{name}: {near_floor.size} cells within 4 ulp of the temperature floor")
    out = {}
    for v in variants:
        p = api.make_params(dt, spec["nsub"], 0.3, spec.get("floor", 0.0), v, api.COOL_COULOMB_TABLE,
                            api.COOL_SCHEME_IMPLICIT if implicit else api.COOL_SCHEME_EXPLICIT)
        api.cool_apply(table, n, api.COOL_F32, d["rho"], d["bsq"], d["theta_e"], d["theta_i"], oe, oi, p,
                       r=d.get("r"), vol=d.get("vol"), d_diag=dg, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        ge, gi = oe.cpu().numpy().astype(np.float64), oi.cpu().numpy().astype(np.float64)
        assert np.isfinite(ge).all() and (ge > 0).all() and (gi > 0).all()
        if idx is not None:
            ge, gi = ge[idx], gi[idx]
        ee, ei = cm.rel_err(ge, rthe), cm.rel_err(gi, rthi)
        if near_floor is not None and near_floor.size:
            # a cell whose gas temperature is within 4 ulp(fp32) of the floor of eq 19 may take either branch (reading C-17: the
            # kernel compares in fp32, the oracle in fp64): it must equal the oracle's answer with the floor test true or false
            for k, alt in ((0, alt_floored), (1, alt_cooled)):
                ea, eia = cm.rel_err(ge[near_floor], alt["theta_e"]), cm.rel_err(gi[near_floor], alt["theta_i"])
                better = np.maximum(ea, eia) < np.maximum(ee[near_floor], ei[near_floor])
                ee[near_floor] = np.where(better, ea, ee[near_floor]); ei[near_floor] = np.where(better, eia, ei[near_floor])
        ce, nact = cm.change_err(ge, rthe, the0)
        label = f"{name} dt={dt:g} {api.VARIANT_NAMES[v]}{' implicit' if implicit else ''}"
        print(f"\n{label}: {'all' if idx is None else 'sampled'} {ge.size} of {n} cells, max rel err e={ee.max():.3e} i={ei.max():.3e}; {nact} cells change by > 1e-3 "
              f"(error of the change {ce:.2e}); kernel {api.cool_last_kernel_name()}, {api.cool_last_launch_count()} launches")
        if implicit:
            # where Lambda is not monotone in Theta_e the implicit equation can have several roots and either is a solution of
            # the scheme (reading C-17): such cells must be rare; tests/test_implicit_gpu.py validates them with the residual
            nbad = int(((ee > gate) | (ei > gate)).sum())
            print(f"  {nbad} cells beyond {gate:g} (other roots)")
            assert nbad <= 2e-5 * ge.size, label
        elif v != api.COOL_V_TEX_HWFILTER:                    # the hardware filter is reported, not gated (8-bit weights)
            assert ee.max() <= gate and ei.max() <= gate, label
            assert ce <= 5e-3 or (near_floor is not None and near_floor.size), label      # the change itself, where there is one
        else:                                                 # reported: the 8-bit filter weights meet the steep K2 interval too
            print(f"  hardware filter: median {np.median(ee):.2e}, 99.9 % quantile {np.quantile(ee, 0.999):.2e}, max {ee.max():.2e}")
            assert np.median(ee) < 1e-5 and np.quantile(ee, 0.999) < 5e-2
        assert np.isfinite(ge).all() and (ge > 0).all() and (gi > 0).all()
        if dg is not None:
            diag = api.cool_diag.from_buffer_copy(dg.cpu().numpy().tobytes()).as_dict()
            rt = 2e-5 if implicit else 2e-6
            if near_floor is not None and near_floor.size:
                rt = 1e-4                                     # a threshold cell's whole loss may go either way
            for k in ("lum_total", "lum_brems", "lum_synch", "lum_compton"):
                if idx is None and v != api.COOL_V_TEX_HWFILTER and (rdiag[k] > 1e-9 * rdiag["lum_total"] or k == "lum_total"):
                    assert diag[k] == pytest.approx(rdiag[k], rel=rt), (label, k)
            if not implicit and v != api.COOL_V_TEX_HWFILTER:
                # event counts: a cell may differ from the oracle only when the compared quantity sits on its threshold
                # (reading C-17): count the oracle's near-threshold cells and allow that many
                near_lim = int((np.abs(ratio / 0.3 - 1.0) <= 1e-5).sum()) if spec["nsub"] == 1 else max(8, int(2e-6 * n))
                assert abs(diag["n_limited"] - rdiag["n_limited"]) <= near_lim, (label, diag["n_limited"], rdiag["n_limited"], near_lim)
                assert abs(diag["n_clamped"] - rdiag["n_clamped"]) <= max(8, int(2e-6 * n)), (label, diag["n_clamped"], rdiag["n_clamped"])
                assert abs(diag["n_floored"] - rdiag["n_floored"]) <= max(8, int(2e-6 * n)), (label, diag["n_floored"], rdiag["n_floored"])
            out["diag"], out["rdiag"] = diag, rdiag
        out["nact"] = nact
    table.destroy()
    return out


def test_config2_fullsize_all_variants(oracle):
    """configs[1]: 256^3 cells, 1 % outliers, table 128^3, every table variant, every cell."""
    out = _run_workload(oracle, "c2", [api.COOL_V_GLOBAL, api.COOL_V_TEX_POINT, api.COOL_V_TEX_HWFILTER])
    assert out["nact"] > 100000


def test_config3_fullsize_density_sweep(oracle):
    """configs[2] at its stated 288 x 192 x 144: MAD-like field, floor on, volume-weighted luminosity, the four density
    normalisations (table rebuilt per rho_scale).  h_floor = 0.117 puts the 5 % noise astride the floor (tests/test_parity_gpu)."""
    for mdot in (1e-6, 1e-4, 1e-2, 0.3):
        rs = synth.rho_scale_for_mdot(mdot)
        out = _run_workload(oracle, "c3", [api.COOL_V_AUTO], units_kw=dict(rho_scale_cgs=rs))
        assert out["diag"]["lum_total"] > 0
    # and once with the floor biting and a time step that moves many cells
    out = _run_workload(oracle, "c3", [api.COOL_V_GLOBAL], dt=50.0, spec_kw=dict(floor=0.117))
    assert out["rdiag"]["n_floored"] > 1000 and out["nact"] > 100000


@pytest.mark.parametrize("m,variants", [(32, [api.COOL_V_SMEM, api.COOL_V_GLOBAL]), (64, [api.COOL_V_GLOBAL]), (128, [api.COOL_V_GLOBAL]),
                                        (256, [api.COOL_V_GLOBAL])])
def test_config4_table_size_sweep(oracle, m, variants):
    """configs[3]: 2^26 log-uniform cells against tables 32^3 (shared memory and the oct layout), 64^3 (octs), 128^3 (quads)
    and 256^3 (plain layout, 64 MiB): one variant per layout, every cell."""
    out = _run_workload(oracle, f"c4-{m}", variants)
    assert out["nact"] > 100000


def test_config5_fullsize_bench_configuration(oracle):
    """configs[4] exactly as bench.py times it: 512^3 MAD-like cells, 3x48^4 + 48^2 tables, nsub=4, luminosity; then the same
    launch at dt = 1 so that many more cells move."""
    out = _run_workload(oracle, "c5", [api.COOL_V_AUTO])
    d = out["diag"]
    assert d["lum_total"] > 0 and d["lum_brems"] + d["lum_synch"] + d["lum_compton"] == pytest.approx(d["lum_total"], rel=1e-5)
    assert out["nact"] > 1000000
    out = _run_workload(oracle, "c5", [api.COOL_V_AUTO], dt=1.0)
    assert out["nact"] > 10000000


def test_s512_fullsize_single_update_3d_step(oracle):
    """The single-update 3-D step at 512^3 (table 128^3, quad layout, 24 warps x 2 stages), and the same with luminosity,
    volume weights and the temperature floor, exactly as bench.py times them."""
    out = _run_workload(oracle, "s512", [api.COOL_V_AUTO])
    assert out["nact"] > 1000000
    out = _run_workload(oracle, "s512f", [api.COOL_V_AUTO])
    assert out["diag"]["lum_total"] > 0          # (h_floor = 0.1 floors no cell of this field: Theta_i + Theta_e = 33 r0/r stays above eq 19)


def test_implicit_fullsize(oracle):
    """The implicit scheme at 512^3 on the 3-D table and on configs[4]'s process tables, as bench.py --scheme implicit times it."""
    _run_workload(oracle, "s512", [api.COOL_V_AUTO], implicit=True, gate=IMPLICIT_GATE)
    _run_workload(oracle, "c5", [api.COOL_V_AUTO], implicit=True, gate=IMPLICIT_GATE)


IMPLICIT_GATE = 1e-5
