"""CPU-side checks of the boundary: the library loads, exports every symbol include/gsp.h
declares, rejects bad arguments, fails loudly without a GPU, and its delay-table builder
(typed independently of the oracle, from rule R3) agrees entry for entry with the oracle
and with the survey's independently computed extents."""
import ctypes
import os

import numpy as np
import pytest

import paper_2110_12749_b200 as gsp
import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_library_exports_every_declared_symbol():
    L = gsp.lib()
    names = gsp.declared_symbols()
    assert {"gsp_plan_create", "gsp_dedisperse", "gsp_plan_destroy", "gsp_dedisperse_host"} <= set(names)
    for n in names:
        assert hasattr(L, n), n
    assert b"sm_100a" in L.gsp_version() and L.gsp_version().startswith(b"libgsp 0.2")
    assert L.gsp_status_string(2) == b"GSP_ERR_TOO_SHORT"


def test_header_has_no_cxx_or_torch_types():
    text = open(os.path.join(os.path.dirname(GOLD), "..", "include", "gsp.h")).read()
    for bad in ("std::", "torch", "at::", "template", "class "):
        assert bad not in text


def test_plan_create_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(gsp.GspError) as ei:
        gsp.Plan(64, 1500.0, -7.8125, 98.304e-6, 8192, 8, 77.5, np.arange(0, 160, 5.0))
    assert ei.value.status == 4  # GSP_ERR_CUDA: no CPU fallback exists


@pytest.mark.parametrize("bad", [
    dict(nchan=0), dict(nsub=0), dict(nsub=7), dict(chan_bw=0.5), dict(chan_bw=0.0),
    dict(f_top=400.0), dict(dt=0.0), dict(dt=-1e-4), dict(downsamp=0), dict(subband_dm=-1.0),
    dict(subband_dm=float("nan")), dict(dm_list=[1.0, -2.0]), dict(dm_list=[float("inf")]),
    dict(dm_list=[]),
])
def test_invalid_arguments_are_rejected(bad):
    a = dict(nchan=64, f_top=1500.0, chan_bw=-7.8125, dt=98.304e-6, nsub=8, subband_dm=77.5,
             dm_list=[0.0, 5.0], downsamp=1)
    a.update(bad)
    with pytest.raises(gsp.GspError) as ei:
        gsp.delay_tables(**a)
    assert ei.value.status == 1


def test_null_pointers_are_rejected():
    L = gsp.lib()
    assert L.gsp_plan_create(None, 64, 1500.0, -7.8, 1e-4, 8192, 8, 0.0, None, 1, 1, 0) == 1
    assert L.gsp_plan_destroy(None) == 0
    assert L.gsp_dedisperse(None, None, None, None) == 1
    assert L.gsp_plan_nout(None) == 0


@pytest.mark.parametrize("name,plan", [("tiny", 0), ("crafts", 0), ("uwb", 0), ("ddplan", 0),
                                       ("ddplan", 1), ("ddplan", 2), ("ddplan", 3)])
def test_library_tables_equal_oracle_tables(oracle_mod, name, plan):
    cfg = workloads.get_config(name)
    a = workloads.plan_args(cfg, plan)
    kw = dict(nchan=a["nchan"], f_top=a["f_top"], chan_bw=a["chan_bw"], dt=a["dt"], nsub=a["nsub"],
              subband_dm=a["subband_dm"], dm_list=a["dm_list"], downsamp=a["downsamp"])
    s1, s2 = gsp.delay_tables(**kw)
    o1, o2 = oracle_mod.delay_tables(**kw)
    np.testing.assert_array_equal(s1, o1)
    np.testing.assert_array_equal(s2, o2)


def test_library_tables_match_survey_extents():
    rows = [l.split() for l in open(os.path.join(GOLD, "table_extents.txt")) if l.strip() and l[0] != "#"]
    for name, plan, H1, H2, nout, sum1, sum2 in rows:
        cfg = workloads.get_config(name)
        a = workloads.plan_args(cfg, int(plan))
        s1, s2 = gsp.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"],
                                  a["subband_dm"], a["dm_list"], a["downsamp"])
        assert int(s1.max()) == int(H1) and int(s2.max()) == int(H2)
        assert (a["nsamp"] - int(H1)) // a["downsamp"] - int(H2) == int(nout)
        if int(sum1) >= 0:
            assert int(s1.sum()) == int(sum1) and int(s2.astype(np.int64).sum()) == int(sum2)


def test_rounding_margin_of_the_tables():
    """Rule R3: on the benchmark tables x + 0.5 never comes closer to an integer than ~1e-6,
    so two independent binary64 evaluations cannot disagree."""
    cfg = workloads.get_config("crafts")
    a = workloads.plan_args(cfg)
    f = a["f_top"] + a["chan_bw"] * np.arange(a["nchan"], dtype=np.float64)
    cps = a["nchan"] // a["nsub"]
    fref = f[::cps]
    x = 4.148808e3 * a["dm_list"][:, None] * (1.0 / fref ** 2 - 1.0 / f[0] ** 2)[None, :] / a["dt"]
    frac = np.abs((x + 0.5) - np.round(x + 0.5))
    assert frac[x > 0].min() > 1e-7
