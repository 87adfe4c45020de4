"""CPU-only checks of the product's host side: the C-ABI library loads and exports every symbol
include/cool.h declares, the host table builder agrees with the oracle node by node, argument
errors are reported (no compute calls that need a GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

import common as cm
from paper_2505_08855_b200 import api, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "cool.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cool_[a-z_]+)\s*\(", hdr))
    assert {"cool_table_create", "cool_apply", "cool_table_destroy", "cool_table_build_host", "cool_apply_host"} <= declared
    L = ctypes.CDLL(api.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(api.EXPORTS)
    assert "sm_100a" in api.cool_version()


def test_struct_layouts_match_header():
    # sizes implied by include/cool.h on LP64
    assert ctypes.sizeof(api.cool_units) == 9 * 8
    assert ctypes.sizeof(api.cool_diag) == 7 * 8
    assert ctypes.sizeof(api.cool_params) == 8 + 8 + 8 + 8 + 8 + 8  # dt, nsub(+pad), f_limit, h_floor, variant+coulomb, scheme(+pad)
    assert ctypes.sizeof(api.cool_cells) == 8 + 8 + 8 * 8 + 8 + 8 + 8  # + shell_cells, lum_shell, flags
    assert ctypes.sizeof(api.cool_table_desc) == 4 + 16 + 16 + 4 + 32 + 32 + 8 + 24 + 8 + 8 + 16 + 16 + 72 + 8 + 12 + 4 + 24 + 24   # + host_coulomb3, nc3 (+pad), c3lo, c3hi


def test_builder_matches_oracle_3d(oracle):
    desc, data, coul = cm.build_tables([64, 64, 64], nc=[64, 64])
    un = cm.oracle_units(oracle, desc)
    T = data[0]
    assert np.isfinite(T).all()
    rng = np.random.default_rng(0)
    ax = [np.linspace(cm.LO3[k], cm.HI3[k], 64) for k in range(3)]
    bad = 0
    for i, j, k in rng.integers(0, 64, size=(1500, 3)):
        ref = oracle.node_total_log10(un, 10 ** ax[0][i], 10 ** ax[1][j], 10 ** ax[2][k])
        assert abs(T[i, j, k] - ref) <= 1e-6 * max(1.0, abs(ref)) + 4e-6       # 1e-6 relative before fp32 rounding
        bad += np.float32(ref) != T[i, j, k]
    assert bad <= 15                      # within 0.5 ulp of round(oracle) except rare rounding ties
    axc = np.linspace(cm.CLO[0], cm.CHI[0], 64)
    for a, b in rng.integers(0, 64, size=(200, 2)):
        assert coul[a, b] == pytest.approx(np.log10(oracle.coulomb_C(10 ** axc[b], 10 ** axc[a])), abs=3e-7)


def test_builder_matches_oracle_4d_and_permuted(oracle):
    desc, data, _ = cm.build_tables([9, 11, 10, 8], nc=[16, 16], axis=[3, 2, 0, 1])
    un = cm.oracle_units(oracle, desc)
    ax = [np.linspace(desc.lo[k], desc.hi[k], desc.n[k]) for k in range(4)]
    rng = np.random.default_rng(1)
    for _ in range(400):
        idx = [rng.integers(0, desc.n[k]) for k in range(4)]
        prim = {desc.axis[k]: 10 ** ax[k][idx[k]] for k in range(4)}
        ref = oracle.node_proc_log10(un, prim[0], prim[1], prim[2], prim[3])
        for p in range(3):
            assert data[p][tuple(idx)] == pytest.approx(ref[p], abs=4e-6)
    # brems table is bit-constant along bsq and Theta_i (it depends on rho and Theta_e only)
    b = data[0]                            # axes (thi, bsq, rho, the)
    assert (b == b[:1, :1]).all()


def test_builder_units_change_table(oracle):
    d1, t1, _ = cm.build_tables([8, 8, 8])
    d2, t2, _ = cm.build_tables([8, 8, 8], units_kw=dict(rho_scale_cgs=1e-9))
    assert not np.allclose(t1[0], t2[0])
    un2 = cm.oracle_units(oracle, d2)
    assert t2[0][3, 4, 5] == pytest.approx(oracle.node_total_log10(un2, 10 ** np.linspace(-6, 0, 8)[3], 10 ** np.linspace(-3, 1.5, 8)[4], 10 ** np.linspace(-8, 0, 8)[5]), abs=4e-6)


def test_builder_and_create_reject_bad_shapes():
    for kw in (dict(n=[1, 4, 4]), dict(axis=[0, 0, 2]), dict(axis=[0, 1, 3]), dict(hi=[-7.0, 1.5, 0.0])):
        args = dict(axis=[0, 1, 2], n=[4, 4, 4], lo=cm.LO3, hi=cm.HI3); args.update(kw)
        d = api.make_desc(args["axis"], args["n"], args["lo"], args["hi"], 1)
        with pytest.raises(api.CoolError) as e:
            api.cool_table_build_host(d)
        assert e.value.status == api.COOL_EINVAL
    d = api.make_desc([0, 1, 2, 3], [4, 4, 4, 4], cm.LO4, cm.HI4, 1)        # 4-D needs nproc = 3
    with pytest.raises(api.CoolError):
        api.cool_table_build_host(d)
    d = api.make_desc([0, 1, 2], [4, 4, 4], cm.LO3, cm.HI3, 1, units=api.default_units(gamma_e=1.0))
    with pytest.raises(api.CoolError):
        api.cool_table_build_host(d)


def test_no_gpu_means_loud_failure():
    """Without a CUDA device cool_table_create must fail with COOL_ECUDA, never fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    desc, data, coul = cm.build_tables([8, 8, 8])
    with pytest.raises(api.CoolError) as e:
        api.cool_table_create(desc, data)
    assert e.value.status == api.COOL_ECUDA
    # the eq 29 correction needs no table: it must fail just as loudly (argument errors come first)
    x = np.ones(8, np.float32)
    with pytest.raises(api.CoolError) as e:
        api.cool_radpress_correct(api.default_units(), 8, api.COOL_F32, x, x, x, 1.0, x)
    assert e.value.status == api.COOL_ECUDA
    with pytest.raises(api.CoolError) as e:
        api.cool_radpress_correct(api.default_units(), 8, api.COOL_F32, x, x, x, -1.0, x)
    assert e.value.status == api.COOL_EINVAL


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2505_08855_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src and "cool_oracle" not in src, fn
    osrc = open(os.path.join(ROOT, "oracle", "cool_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "#include \"cool" not in osrc and "import paper_2505_08855_b200" not in osrc and "from paper_2505_08855_b200" not in osrc
