"""gsp_dedisperse_static — the entry point for callers that are not allowed to allocate device memory.

Who that is: a telescope backend thread that keeps recording on other streams (cudaMalloc / cudaFree
synchronise the whole device and would stall them), a process whose device memory was handed out in full at
start-up by some other owner (a framework's pool, a fixed arena), or any code running after its project's
"no allocation past initialisation" line.  They cannot create a gsp_plan (it allocates its tables and its
subband workspace), so the library gives them one plan-free call that keeps the subband intermediate in a
fixed 16 MiB array inside the library image and calls no cudaMalloc / cudaFree at all.

What is checked here: the call's output equals the existing path's (gsp_plan_create + gsp_dedisperse with the
kernels the library picks by itself) — bit for bit on uint8 input, within the suite's float32 tolerance on
float32 input — on TWO calls in a row with different shapes, because every call works in the same array and
finds the previous call's intermediate still in it.  Problems beyond the array's size must be refused with
GSP_ERR_TOO_LARGE before any GPU work.

This file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a
failure here must not hide the parity tests.  It passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

import paper_2110_12749_b200 as gsp

F32_TOL = 1e-5          # the tolerance of tests/test_gpu_parity.py (reading A13)
SENTINEL = -12345.0


def _args(nchan, nsub, ndm, ds, nsamp, dtype, seed, dm_hi=200.0, f_top=1500.0, bw=500.0, dt=98.304e-6):
    rng = np.random.default_rng(seed)
    dms = np.sort(rng.uniform(0.0, dm_hi, size=ndm))
    a = dict(nchan=nchan, f_top=f_top, chan_bw=-bw / nchan, dt=dt, nsamp=nsamp, nsub=nsub,
             subband_dm=float(dms.mean()), dm_list=dms, downsamp=ds, dtype=dtype)
    if dtype == "u8":
        x = rng.integers(0, 256, size=(nsamp, nchan), dtype=np.uint8)
    else:
        x = rng.normal(10.0, 3.0, size=(nsamp, nchan)).astype(np.float32)
    return a, x


def _existing_path(a, x_dev):
    """What a caller who MAY allocate gets: a plan and gsp_dedisperse, kernels chosen by the library."""
    import torch
    with gsp.Plan(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsamp"], a["nsub"], a["subband_dm"],
                  a["dm_list"], a["downsamp"], a["dtype"]) as plan:
        out = torch.full((plan.ndm, plan.out_pitch), SENTINEL, dtype=torch.float32, device="cuda")
        plan.dedisperse(x_dev, out, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        return out.cpu().numpy()[:, : plan.nout], plan.nout, plan.out_pitch, plan.H1, plan.H2


def _static_path(a, x_dev, out_pitch):
    """What a caller who may NOT allocate does: tables on the host (gsp_delay_tables makes no CUDA call),
    copied into memory the caller already owns — here torch tensors stand in for that memory — then the one
    plan-free call.  Returns (output rows incl. padding, nout)."""
    import torch
    s1, s2 = gsp.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"], a["subband_dm"],
                              a["dm_list"], a["downsamp"])
    h1, h2 = int(s1.max()), int(s2.max())
    nout = (a["nsamp"] - h1) // a["downsamp"] - h2
    ndm = len(a["dm_list"])
    d_s1, d_s2 = torch.from_numpy(s1).cuda(), torch.from_numpy(s2).cuda()
    out = torch.full((ndm, out_pitch), SENTINEL, dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    gsp.dedisperse_static(x_dev, a["dtype"], a["nsamp"], a["nchan"], a["nsub"], ndm, a["downsamp"], d_s1, d_s2,
                          h1, h2, out, out_pitch, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out.cpu().numpy(), nout


def _compare(a, x, exact):
    import torch
    x_dev = torch.from_numpy(x).cuda()
    want, nout, pitch, h1, h2 = _existing_path(a, x_dev)
    got_full, nout_s = _static_path(a, x_dev, pitch)
    assert nout_s == nout
    assert np.all(got_full[:, nout:] == SENTINEL), "columns past nout must stay untouched"
    got = got_full[:, :nout]
    if exact:
        bad = np.flatnonzero(got != want)
        assert bad.size == 0, f"{bad.size} mismatches, first at {np.unravel_index(bad[0], got.shape)}"
    else:
        rms = np.sqrt((want.astype(np.float64) ** 2).mean(axis=1, keepdims=True))
        den = np.maximum(np.abs(want), rms)
        den[den == 0] = 1.0
        assert float((np.abs(got.astype(np.float64) - want) / den).max()) <= F32_TOL
    return got


@pytest.mark.gpu
def test_static_call_equals_the_plan_path_on_two_calls_in_a_row_u8():
    # call 1 and call 2 differ in every size, so call 2 finds call 1's intermediate (other row length,
    # other values) in the shared array; call 3 repeats call 1 and must reproduce it exactly
    a1, x1 = _args(nchan=64, nsub=8, ndm=37, ds=1, nsamp=9001, dtype="u8", seed=1)
    a2, x2 = _args(nchan=96, nsub=12, ndm=20, ds=3, nsamp=12345, dtype="u8", seed=2)
    first = _compare(a1, x1, exact=True)
    _compare(a2, x2, exact=True)
    again = _compare(a1, x1, exact=True)
    np.testing.assert_array_equal(first, again)


@pytest.mark.gpu
def test_static_call_equals_the_plan_path_on_two_calls_in_a_row_f32():
    a1, x1 = _args(nchan=128, nsub=16, ndm=33, ds=2, nsamp=20011, dtype="f32", seed=3)
    a2, x2 = _args(nchan=64, nsub=8, ndm=9, ds=1, nsamp=7000, dtype="f32", seed=4)
    _compare(a1, x1, exact=False)
    _compare(a2, x2, exact=False)


@pytest.mark.gpu
def test_static_call_on_a_survey_shaped_block_near_the_size_limit():
    # 4096 channels / 64 subbands like the CRAFTS-like beam, a time block that nearly fills the 16 MiB array
    # (64 subbands x ~65000 samples x 4 bytes), against the library's product kernels; twice in a row
    nsamp = 65000
    a, x = _args(nchan=4096, nsub=64, ndm=48, ds=1, nsamp=nsamp, dtype="u8", seed=5, dm_hi=60.0,
                 f_top=1499.9, bw=500.0)
    s1, _ = gsp.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"], a["subband_dm"],
                             a["dm_list"], 1)
    need = 64 * (nsamp - int(s1.max())) * 4
    assert 0.9 * gsp.static_workspace_bytes() < need <= gsp.static_workspace_bytes()
    first = _compare(a, x, exact=True)
    again = _compare(a, x, exact=True)
    np.testing.assert_array_equal(first, again)


@pytest.mark.gpu
def test_static_call_refuses_a_problem_beyond_its_array_on_the_gpu_box():
    import torch
    a, _ = _args(nchan=64, nsub=8, ndm=4, ds=1, nsamp=1 << 20, dtype="u8", seed=6)   # 8 x ~2^20 x 4 B = 32 MiB
    s1, s2 = gsp.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"], a["subband_dm"],
                              a["dm_list"], 1)
    x = torch.zeros((a["nsamp"], a["nchan"]), dtype=torch.uint8, device="cuda")
    out = torch.full((4, a["nsamp"]), SENTINEL, dtype=torch.float32, device="cuda")
    with pytest.raises(gsp.GspError) as err:
        gsp.dedisperse_static(x, "u8", a["nsamp"], 64, 8, 4, 1, torch.from_numpy(s1).cuda(),
                              torch.from_numpy(s2).cuda(), int(s1.max()), int(s2.max()), out, a["nsamp"],
                              torch.cuda.current_stream().cuda_stream)
    assert err.value.status == 5 and "GSP_ERR_TOO_LARGE" in str(err.value)
    torch.cuda.synchronize()
    assert bool((out == SENTINEL).all()), "a refused call must not touch the output"


def test_static_call_checks_sizes_before_any_gpu_work():
    """Host-only: the refusals are plain arithmetic made before the first CUDA call, so they can be checked
    without a device (the addresses below are never dereferenced)."""
    assert gsp.static_workspace_bytes() == 16 << 20
    fake = 0x1000
    L = gsp.lib()
    assert L.gsp_status_string(5) == b"GSP_ERR_TOO_LARGE"

    def call(nsamp=10000, nchan=64, nsub=8, ndm=4, ds=1, h1=10, h2=20, pitch=None, d_in=fake, dtype=0):
        pitch = nsamp if pitch is None else pitch
        return L.gsp_dedisperse_static(d_in, dtype, nsamp, nchan, nsub, ndm, ds, fake, fake, h1, h2, fake, pitch, None)

    limit = (16 << 20) // 4 // 8                          # n1d that exactly fills the array with 8 subbands
    assert call(nsamp=limit + 10 + 1) == 5                # one sample too many: TOO_LARGE
    assert call(nsamp=1 << 24) == 5
    assert call(nsamp=25) == 2                            # nout <= 0: TOO_SHORT
    assert call(d_in=None) == 1                           # null pointer
    assert call(nsub=7) == 1                              # nsub does not divide nchan
    assert call(dtype=2) == 1                             # unknown element type
    assert call(pitch=100) == 1                           # out_pitch < nout
    assert call(ndm=70000) == 1                           # beyond the launch grid
