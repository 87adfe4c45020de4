"""cool_apply_noalloc (include/cool.h): the step with its scratch memory in a static device array, for callers that cannot
call cudaMalloc.  Its output must equal cool_apply's (same kernels, same launch shapes), on two calls in a row that share
the scratch array, the second on other inputs so that the first call's leftovers are really there.

Collected last on purpose (the suite runs with pytest -x)."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2505_08855_b200 import api, synth

import common as cm

pytestmark = pytest.mark.gpu

TOL = {np.float32: 1e-5, np.float64: 1e-12}          # the parity bars of tests/test_parity_gpu.py
LUM_TOL = 2e-6                                       # luminosity sums (tests/test_fullsize_gpu.py)


def _device_fields(fields, dtype, keys):
    import torch
    tdt = torch.float32 if dtype == np.float32 else torch.float64
    return {k: torch.from_numpy(np.ascontiguousarray(fields[k], dtype=dtype)).to("cuda:0", tdt) for k in keys}


def _run(entry, table, d, dtype, params, use_r, use_vol):
    """One call of `entry` (api.cool_apply or api.cool_apply_noalloc) on device arrays -> (theta_e', theta_i', diag, flags, launches)."""
    import torch
    n = d["rho"].numel()
    cdt = api.COOL_F32 if dtype == np.float32 else api.COOL_F64
    the_o, thi_o = torch.empty_like(d["theta_e"]), torch.empty_like(d["theta_i"])
    d_diag = torch.full((api.DIAG_BYTES,), 255, dtype=torch.uint8, device="cuda:0")          # must be overwritten
    flags = torch.full((n,), 255, dtype=torch.uint8, device="cuda:0")
    entry(table, n, cdt, d["rho"], d["bsq"], d["theta_e"], d["theta_i"], the_o, thi_o, params,
          r=d["r"] if use_r else None, vol=d["vol"] if use_vol else None, d_diag=d_diag,
          stream=torch.cuda.current_stream().cuda_stream, flags=flags)
    launches = api.cool_last_launch_count()
    torch.cuda.synchronize()
    diag = api.cool_diag.from_buffer_copy(d_diag.cpu().numpy().tobytes()).as_dict()
    return the_o.cpu().numpy().astype(np.float64), thi_o.cpu().numpy().astype(np.float64), diag, flags.cpu().numpy(), launches


CASES = [
    # name, table shape, Coulomb table, dtype, dt, nsub, floor, first field, second field (r, theta, phi)
    ("4d_substeps_f32", [20, 22, 18, 16], [24, 24], np.float32, 1.0, 4, 0.0, (64, 48, 40), (40, 33, 29)),      # partials + ticket + precise-pass lists
    ("3d_single_f32", [48, 48, 48], [32, 32], np.float32, 1e-2, 1, 0.1, (64, 48, 40), (37, 31, 23)),           # partials + ticket
    ("3d_substeps_f32", [48, 48, 48], [32, 32], np.float32, 1.0, 3, 0.0, (64, 48, 40), (37, 31, 23)),          # lists of the 3-D step
    ("3d_single_f64", [32, 32, 32], [32, 32], np.float64, 1e-2, 2, 0.1, (48, 32, 24), (25, 17, 13)),           # the fp64 kernel's partials
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_noalloc_matches_cool_apply_on_two_calls_in_a_row(case):
    import torch
    name, n, nc, dtype, dt, nsub, floor, shape1, shape2 = case
    desc, data, coul = cm.build_tables(n, nc=nc)
    table = api.cool_table_create(desc, data, coul, device=0)
    try:
        params = api.make_params(dt, nsub, 0.3, floor, api.COOL_V_AUTO, api.COOL_COULOMB_TABLE)
        keys = ("rho", "bsq", "theta_e", "theta_i", "r", "vol")
        batches = []
        for k, shp in enumerate((shape1, shape2)):
            f = synth.mad_like_cells(*shp, dtype=dtype, config=40 + k)
            batches.append(_device_fields(f, dtype, keys))
        use_r, use_vol = floor > 0.0, True
        ref = [_run(api.cool_apply, table, d, dtype, params, use_r, use_vol) for d in batches]
        # warm-up of the new entry point (resolves the scratch address, loads its kernels), then the two calls in a row; the
        # device's free memory must not move between them: nothing is allocated
        api.cool_apply_noalloc(table, 0, api.COOL_F32 if dtype == np.float32 else api.COOL_F64, batches[0]["rho"], batches[0]["bsq"],
                               batches[0]["theta_e"], batches[0]["theta_i"], batches[0]["theta_e"], batches[0]["theta_i"], params)
        got = [_run(api.cool_apply_noalloc, table, batches[0], dtype, params, use_r, use_vol)]
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info(0)[0]
        got.append(_run(api.cool_apply_noalloc, table, batches[1], dtype, params, use_r, use_vol))
        got.append(_run(api.cool_apply_noalloc, table, batches[0], dtype, params, use_r, use_vol))      # and back: the larger batch after the smaller
        torch.cuda.synchronize()
        free1 = torch.cuda.mem_get_info(0)[0]
        ref.append(ref[0])
        active = 0
        for k, (g, r) in enumerate(zip(got, ref)):
            e = max(cm.rel_err(g[0], r[0]).max(), cm.rel_err(g[1], r[1]).max())
            assert e <= TOL[dtype], f"{name} call {k}: max rel err {e:.3g} vs cool_apply"
            assert np.array_equal(g[0], r[0]) and np.array_equal(g[1], r[1]), f"{name} call {k}: same kernels, same launch shape: bit-identical outputs expected"
            assert np.array_equal(g[3], r[3]), f"{name} call {k}: per-cell flags differ"
            assert g[4] == r[4], f"{name} call {k}: {g[4]} launches vs {r[4]}"
            for key in ("lum_total", "lum_brems", "lum_synch", "lum_compton"):
                assert abs(g[2][key] - r[2][key]) <= LUM_TOL * abs(r[2]["lum_total"]), f"{name} call {k}: {key} {g[2][key]} vs {r[2][key]}"
            for key in ("n_limited", "n_floored", "n_clamped"):
                assert g[2][key] == r[2][key], f"{name} call {k}: {key}"
            active += int((g[3] & 8).sum())
        # anti-vacuity: the step did something, and the case that is there for the lists really listed cells
        assert ref[0][2]["lum_total"] > 0.0
        if name in ("4d_substeps_f32", "3d_substeps_f32"):
            assert got[0][4] == 2 and active > 0, f"{name}: expected the precise pass to run ({got[0][4]} launches, {active} cells)"
        assert free1 == free0, f"{name}: device free memory moved by {free0 - free1} bytes across two cool_apply_noalloc calls"
    finally:
        table.destroy()


def test_noalloc_rejects_what_it_cannot_hold():
    import torch
    desc, data, coul = cm.build_tables([16, 16, 16], nc=[16, 16])
    table = api.cool_table_create(desc, data, coul, device=0)
    try:
        x = torch.ones(1024, dtype=torch.float32, device="cuda:0")
        y = torch.empty_like(x)
        params = api.make_params(1e-3, 1, 0.3, 0.0, api.COOL_V_AUTO, api.COOL_COULOMB_TABLE)
        with pytest.raises(api.CoolError) as ei:             # beyond the maximum: nothing is launched (the arrays hold 1024 cells)
            api.cool_apply_noalloc(table, api.COOL_NOALLOC_MAX_CELLS + 1, api.COOL_F32, x, x, x, x, y, y, params)
        assert "COOL_NOALLOC_MAX_CELLS" in str(ei.value)
        torch.cuda.synchronize()
        # the radial profile needs a growing workspace: refused
        c = api._cells(1024, api.COOL_F32, x, x, x, x, y, y, None, None, 128, torch.zeros(32, dtype=torch.float64, device="cuda:0"), None)
        d_diag = torch.zeros(api.DIAG_BYTES, dtype=torch.uint8, device="cuda:0")
        import ctypes as C
        rc = api.lib().cool_apply_noalloc(table.handle, C.byref(c), C.byref(params), api._ptr(d_diag), None)
        assert rc != 0 and b"lum_shell" in api.lib().cool_last_error()
    finally:
        table.destroy()


def test_noalloc_at_the_maximum_size():
    """the largest batch it takes: sub-stepped 4-D step, so partials, ticket and the largest lists"""
    import torch
    n = api.COOL_NOALLOC_MAX_CELLS
    desc, data, coul = cm.build_tables([20, 22, 18, 16], nc=[24, 24])
    table = api.cool_table_create(desc, data, coul, device=0)
    try:
        f = synth.mad_like_cells(256, 256, 256, dtype=np.float32, config=42)
        d = _device_fields(f, np.float32, ("rho", "bsq", "theta_e", "theta_i", "r", "vol"))
        assert d["rho"].numel() == n
        params = api.make_params(1.0, 4, 0.3, 0.0, api.COOL_V_AUTO, api.COOL_COULOMB_TABLE)
        ref = _run(api.cool_apply, table, d, np.float32, params, False, True)
        got = _run(api.cool_apply_noalloc, table, d, np.float32, params, False, True)
        assert np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1])
        assert abs(got[2]["lum_total"] - ref[2]["lum_total"]) <= LUM_TOL * abs(ref[2]["lum_total"])
        assert got[4] == ref[4] == 2 and int((got[3] & 8).sum()) > 0
    finally:
        table.destroy()
