"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (same workload
recipes, same tables, same cool_apply call), on sampled outputs the oracle computes one by one,
plus properties that hold at any size."""
import numpy as np
import pytest

import bench
import common as cm
from paper_2505_08855_b200 import api, synth

pytestmark = pytest.mark.gpu


def _run_workload(oracle, name, variants, nsample=20000, implicit=False):
    import torch
    spec = bench.workload_spec(name)
    axis, lo, hi = bench.table_ranges(spec["n"])
    desc = api.make_desc(axis, spec["n"], lo, hi, 1 if len(spec["n"]) == 3 else 3, nc=spec["nc"], clo=cm.CLO, chi=cm.CHI)
    data, coul = api.cool_table_build_host(desc, want_coulomb=True)
    table = api.cool_table_create(desc, data, coul)
    otab, un = cm.oracle_table(oracle, desc, data, coul), cm.oracle_units(oracle, desc)
    f = bench.make_fields(spec)
    n = f["rho"].size
    dev = torch.device("cuda:0")
    keys = ["rho", "bsq", "theta_e", "theta_i"] + (["vol"] if spec.get("vol") else []) + (["r"] if spec.get("floor") else [])
    d = {k: torch.from_numpy(f[k]).to(dev) for k in keys}
    oe = torch.empty(n, dtype=torch.float32, device=dev); oi = torch.empty_like(oe)
    dg = torch.zeros(api.DIAG_BYTES, dtype=torch.uint8, device=dev) if spec["diag"] else None
    idx = np.sort(np.random.default_rng(11).choice(n, nsample, replace=False))
    sub = {k: f[k][idx] for k in keys}
    ostep = cm.oracle_step_implicit if implicit else cm.oracle_step
    ref = ostep(oracle, otab, un, sub, spec["dt"], nsub=spec["nsub"], h_floor=spec.get("floor", 0.0),
                use_r=bool(spec.get("floor")), use_vol=bool(spec.get("vol")))
    tol = 5e-5 if implicit else 1e-5
    out = {}
    for v in variants:
        p = api.make_params(spec["dt"], spec["nsub"], 0.3, spec.get("floor", 0.0), v, api.COOL_COULOMB_TABLE,
                            api.COOL_SCHEME_IMPLICIT if implicit else api.COOL_SCHEME_EXPLICIT)
        api.cool_apply(table, n, api.COOL_F32, d["rho"], d["bsq"], d["theta_e"], d["theta_i"], oe, oi, p,
                       r=d.get("r"), vol=d.get("vol"), d_diag=dg, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        ge, gi = oe.cpu().numpy(), oi.cpu().numpy()
        ee, ei = cm.rel_err(ge[idx], ref["theta_e"]).max(), cm.rel_err(gi[idx], ref["theta_i"]).max()
        gated = v != api.COOL_V_TEX_HWFILTER
        print(f"\n{name} {api.VARIANT_NAMES[v]}: sampled max rel err e={ee:.3e} i={ei:.3e}")
        if gated:
            assert ee <= tol and ei <= tol, (name, api.VARIANT_NAMES[v], ee, ei)
        else:
            assert ee < 5e-2
        # any-size properties: finite, positive, electrons never lose more than 1-(1-2f)^nsub
        assert np.isfinite(ge).all() and (ge > 0).all() and (gi > 0).all()
        if not implicit:
            assert (ge >= f["theta_e"] * (0.4 ** spec["nsub"]) * (1 - 1e-6)).all()
        if dg is not None:
            diag = api.cool_diag.from_buffer_copy(dg.cpu().numpy().tobytes()).as_dict()
            mr = 9.1093837015e-28 / 1.67262192369e-24
            w = f["vol"].astype(np.float64) if spec.get("vol") else 1.0
            drop = (f["rho"].astype(np.float64) * ((f["theta_e"].astype(np.float64) + f["theta_i"]) - (ge.astype(np.float64) + gi)) * w).sum() * mr * 1.5 / spec["dt"]
            # energy only leaves through radiation (fp32 rounding of Theta' limits the agreement)
            assert diag["lum_total"] == pytest.approx(drop, rel=2e-2)
            out["diag"] = diag
    table.destroy()
    return out


def test_config2_fullsize_all_variants(oracle):
    """configs[1]: 256^3 cells, 1 % outliers, table 128^3, every table variant."""
    _run_workload(oracle, "c2", [api.COOL_V_GLOBAL, api.COOL_V_TEX_POINT, api.COOL_V_TEX_HWFILTER])


def test_config5_fullsize_bench_configuration(oracle):
    """configs[4] exactly as bench.py times it: 512^3 MAD-like cells, 3x48^4 + 48^2 tables, nsub=4, luminosity."""
    out = _run_workload(oracle, "c5", [api.COOL_V_AUTO])
    d = out["diag"]
    assert d["lum_total"] > 0 and d["lum_brems"] + d["lum_synch"] + d["lum_compton"] == pytest.approx(d["lum_total"], rel=1e-5)


def test_s512_fullsize_single_update_3d_step(oracle):
    """The single-update 3-D step at 512^3 (table 128^3, quad layout, 24 warps x 2 stages) and the same with luminosity,
    volume weights and the temperature floor, exactly as bench.py times them."""
    _run_workload(oracle, "s512", [api.COOL_V_AUTO])
    out = _run_workload(oracle, "s512f", [api.COOL_V_AUTO])
    assert out["diag"]["lum_total"] > 0          # (h_floor = 0.1 floors no cell of this field: Theta_i + Theta_e = 33 r0/r stays above eq 19)


def test_implicit_fullsize(oracle):
    """The implicit scheme at 512^3 on the 3-D table and on configs[4]'s process tables, as bench.py --scheme implicit times it."""
    _run_workload(oracle, "s512", [api.COOL_V_AUTO], implicit=True)
    _run_workload(oracle, "c5", [api.COOL_V_AUTO], implicit=True)
