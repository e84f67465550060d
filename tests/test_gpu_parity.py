"""GPU parity: libgsp (through the C ABI binding) against the CPU oracle, element by element.

uint8 input must be bit-exact (integer sums < 2^24 are exact in int32 and float32);
float32 input must satisfy  max |g - r| / max(|r|, rms_u(r_d)) <= 1e-5  per DM row
(reading A13) against the oracle that sums in binary64.
"""
import numpy as np
import pytest
import torch

import paper_2110_12749_b200 as gsp
import workloads

pytestmark = pytest.mark.gpu

F32_TOL = 1e-5
# (stage-1 impl, stage-2 impl): Algorithm 2 applied twice; the tiled kernels bench.py times; and
# the tiled stage 1 feeding the generic stage 2 (its int32 workspace format)
IMPLS = [(gsp.GSP_IMPL_GENERIC, gsp.GSP_IMPL_GENERIC), (gsp.GSP_IMPL_AUTO, gsp.GSP_IMPL_AUTO),
         (gsp.GSP_IMPL_AUTO, gsp.GSP_IMPL_GENERIC), (gsp.GSP_IMPL_GENERIC, gsp.GSP_IMPL_AUTO),
         (gsp.GSP_IMPL_WINDOWED, gsp.GSP_IMPL_AUTO)]


def _set(plan, impl):
    try:
        plan.set_impl(1, impl[0])
    except gsp.GspError:
        if impl[0] != gsp.GSP_IMPL_WINDOWED:
            raise
        pytest.skip("windowed stage-1 kernel does not cover this shape")
    plan.set_impl(2, impl[1])


def _run(plan, x_dev):
    out = torch.full((plan.ndm, plan.out_pitch), -12345.0, dtype=torch.float32, device="cuda")
    plan.dedisperse(x_dev, out, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    assert np.all(res[:, plan.nout:] == -12345.0), "padding columns must not be written"
    return res[:, : plan.nout]


def _f32_err(g, r):
    rms = np.sqrt((r.astype(np.float64) ** 2).mean(axis=1, keepdims=True))
    den = np.maximum(np.abs(r), rms)
    den[den == 0] = 1.0
    return float((np.abs(g.astype(np.float64) - r) / den).max())


def _oracle_tables(plan, oracle_mod):
    """The ORACLE's delay tables for the plan's arguments; the library's own tables must equal them entry
    for entry (they are typed independently from rule R3), and it is the oracle's that the oracle is fed."""
    a = plan.args
    s1, s2 = oracle_mod.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"], a["subband_dm"],
                                     a["dm_list"], a["downsamp"])
    np.testing.assert_array_equal(plan.stage1_shifts, s1)
    np.testing.assert_array_equal(plan.stage2_shifts, s2)
    return s1, s2


def _oracle_tables_args(a, oracle_mod):
    return oracle_mod.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"], a["subband_dm"],
                                   a["dm_list"], a["downsamp"])


def _check(plan, x_np, oracle_mod, ds, exact):
    assert ds == plan.args["downsamp"]
    s1, s2 = _oracle_tables(plan, oracle_mod)
    want = oracle_mod.dedisperse(x_np, s1, s2, ds, nthreads=oracle_mod.max_threads())
    assert want.shape == (plan.ndm, plan.nout)
    got = _run(plan, torch.from_numpy(x_np).cuda())
    if exact:
        bad = np.flatnonzero(got != want)
        assert bad.size == 0, f"{bad.size} mismatches, first at {np.unravel_index(bad[0], got.shape)}"
    else:
        assert _f32_err(got, want) <= F32_TOL
    return got, want


def _mkplan(a, nsamp=None, **over):
    kw = dict(a)
    kw.update(over)
    if nsamp is not None:
        kw["nsamp"] = nsamp
    plan = gsp.Plan(kw["nchan"], kw["f_top"], kw["chan_bw"], kw["dt"], kw["nsamp"], kw["nsub"],
                    kw["subband_dm"], kw["dm_list"], kw["downsamp"], kw["dtype"])
    plan.args = kw
    return plan


# --------------------------------------------------------------------------- config 1
@pytest.mark.parametrize("impl2", IMPLS, ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
def test_tiny_config_bit_exact(oracle_mod, impl2):
    cfg = workloads.get_config("tiny")
    a = workloads.plan_args(cfg)
    x = workloads.make_filterbank(cfg).numpy()
    with _mkplan(a) as plan:
        _set(plan, impl2)
        np.testing.assert_array_equal(plan.stage1_shifts, oracle_mod.delay_tables(
            a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"], a["subband_dm"], a["dm_list"], 1)[0])
        got, _ = _check(plan, x, oracle_mod, 1, exact=True)
        assert plan.nout == 4982
    # the noise-free injected pulse peaks at DM 100 and its arrival sample (pin P11, on the GPU)
    xp = workloads.make_filterbank(cfg, noise=False).numpy()
    with _mkplan(a) as plan:
        _set(plan, impl2)
        y = _run(plan, torch.from_numpy(xp).cuda())
        d, u = np.unravel_index(np.argmax(y), y.shape)
        assert (d, u, y.max()) == (20, 3000, 320.0)


def test_tiled_stage2_is_selected_for_the_benchmark_shapes():
    cfg = workloads.get_config("crafts")
    a = workloads.plan_args(cfg, nsamp=1 << 17)
    with _mkplan(a) as plan:
        assert plan.get_impl(2) == gsp.GSP_IMPL_TILED
        assert plan.get_impl(1) == gsp.GSP_IMPL_TILED


# --------------------------------------------------------------------------- ragged / edge shapes
@pytest.mark.parametrize("impl2", IMPLS, ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
@pytest.mark.parametrize("case", [
    dict(nchan=64, nsub=8, ndm=37, ds=1, nsamp=9001),      # ndm not a multiple of any DM block
    dict(nchan=64, nsub=8, ndm=5, ds=2, nsamp=9000),
    dict(nchan=96, nsub=12, ndm=70, ds=3, nsamp=12345),    # non power-of-two downsamp
    dict(nchan=128, nsub=4, ndm=33, ds=4, nsamp=20011),
    dict(nchan=32, nsub=32, ndm=9, ds=1, nsamp=5000),      # one channel per subband
    dict(nchan=32, nsub=1, ndm=9, ds=1, nsamp=5000),       # one subband (generic only)
    dict(nchan=60, nsub=6, ndm=3, ds=1, nsamp=7000),       # nsub not a multiple of 4
    dict(nchan=64, nsub=8, ndm=1, ds=8, nsamp=30000),
])
def test_ragged_shapes_u8_bit_exact(oracle_mod, impl2, case):
    rng = np.random.default_rng(case["nsamp"])
    dms = np.sort(rng.uniform(0, 200, size=case["ndm"]))
    a = dict(nchan=case["nchan"], f_top=1500.0, chan_bw=-500.0 / case["nchan"], dt=98.304e-6,
             nsamp=case["nsamp"], nsub=case["nsub"], subband_dm=float(dms.mean()), dm_list=dms,
             downsamp=case["ds"], dtype="u8")
    x = rng.integers(0, 256, size=(case["nsamp"], case["nchan"]), dtype=np.uint8)
    with _mkplan(a) as plan:
        _set(plan, impl2)
        _check(plan, x, oracle_mod, case["ds"], exact=True)


# --------------------------------------------------------------------------- wide shifts (low band)
@pytest.mark.parametrize("impl2", IMPLS, ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
@pytest.mark.parametrize("case", [
    # 400 -> 272 MHz: a channel's shift differs from its neighbour's by 100-900 rows
    dict(nchan=256, nsub=8, ds=1, sdm=30.0, nsamp=30000, want="long_mid"),   # cps 32: common stream + per-slice streams, two CTAs per SM
    dict(nchan=256, nsub=8, ds=1, sdm=100.0, nsamp=30000, want="long_big"),  # cps 32: per-slice streams, rings up to 200 KB
    dict(nchan=128, nsub=8, ds=4, sdm=90.0, nsamp=30000, want="long_big"),   # cps 16: one slice, chunks of 1024 rows
    dict(nchan=128, nsub=8, ds=2, sdm=40.0, nsamp=20011, want="long_mid"),   # cps 16
    dict(nchan=256, nsub=4, ds=1, sdm=25.0, nsamp=30000, want="long_mid"),   # cps 64: four slices, per-slice streams
    dict(nchan=256, nsub=4, ds=2, sdm=60.0, nsamp=30011, want="long_big"),   # cps 64: per-slice streams, one CTA per SM
    dict(nchan=256, nsub=4, ds=2, sdm=140.0, nsamp=40011, want="mid"),     # cps 64, wide kernel, clusters of 4
    dict(nchan=256, nsub=8, ds=1, sdm=250.0, nsamp=45000, want="big"),     # wide ring > half the shared memory
    dict(nchan=256, nsub=8, ds=1, sdm=640.0, nsamp=70000, want="windowed"),  # too wide for any ring
], ids=lambda c: f"{c['nchan']}ch_{c['nsub']}sub_ds{c['ds']}_sdm{c['sdm']:g}_{c['want']}")
def test_wide_shift_groups_u8_bit_exact(oracle_mod, impl2, case):
    """Subbands whose stage-1 shifts exceed the standard channel-major ring stream through its long-ring
    instantiation (one CTA per subband), the wide kernel (time-major ring, clusters over 16-channel groups)
    or, beyond that, the windowed kernel."""
    rng = np.random.default_rng(case["nsamp"])
    dms = np.sort(rng.uniform(0, 12, size=21))
    a = dict(nchan=case["nchan"], f_top=400.0, chan_bw=-128.0 / case["nchan"], dt=98.304e-6,
             nsamp=case["nsamp"], nsub=case["nsub"], subband_dm=case["sdm"], dm_list=dms,
             downsamp=case["ds"], dtype="u8")
    x = rng.integers(0, 256, size=(case["nsamp"], case["nchan"]), dtype=np.uint8)
    with _mkplan(a) as plan:
        _set(plan, impl2)
        if impl2[0] == gsp.GSP_IMPL_AUTO:
            ring, mid, big, win, _, lmid, lbig = plan.stage1_split
            assert plan.get_impl(1) == gsp.GSP_IMPL_TILED
            assert {"mid": mid > 0, "big": big > 0, "windowed": win > 0 and mid + big < case["nsub"],
                    "long_mid": lmid > 0, "long_big": lbig > 0}[case["want"]], (ring, mid, big, win, lmid, lbig)
        _check(plan, x, oracle_mod, case["ds"], exact=True)


@pytest.mark.parametrize("impl2", IMPLS, ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
def test_unsorted_and_duplicate_dm_list(oracle_mod, impl2):
    rng = np.random.default_rng(5)
    dms = np.array([150.0, 0.0, 75.5, 150.0, 3.0, 199.0, 42.0, 42.0, 7.0, 120.0, 0.0])
    a = dict(nchan=64, f_top=1500.0, chan_bw=-7.8125, dt=98.304e-6, nsamp=12000, nsub=8,
             subband_dm=60.0, dm_list=dms, downsamp=1, dtype="u8")
    x = rng.integers(0, 256, size=(12000, 64), dtype=np.uint8)
    with _mkplan(a) as plan:
        _set(plan, impl2)
        got, _ = _check(plan, x, oracle_mod, 1, exact=True)
        np.testing.assert_array_equal(got[0], got[3])
        np.testing.assert_array_equal(got[1], got[10])


@pytest.mark.parametrize("impl2", IMPLS, ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
def test_saturated_input_max_sums(oracle_mod, impl2):
    """All samples 255: the 16-bit partial sums reach their bound 4*cps*255*ds exactly."""
    for nchan, nsub, ds in ((256, 4, 1), (256, 8, 2), (4096, 64, 1)):
        nsamp = 6000
        dms = np.arange(0, 40, 1.0)
        a = dict(nchan=nchan, f_top=1500.0, chan_bw=-500.0 / nchan, dt=98.304e-6, nsamp=nsamp,
                 nsub=nsub, subband_dm=20.0, dm_list=dms, downsamp=ds, dtype="u8")
        x = np.full((nsamp, nchan), 255, dtype=np.uint8)
        with _mkplan(a) as plan:
            _set(plan, impl2)
            got = _run(plan, torch.from_numpy(x).cuda())
            assert np.all(got == np.float32(255 * nchan))


def test_minimum_length_input_single_output(oracle_mod):
    cfg = workloads.get_config("tiny")
    a = workloads.plan_args(cfg)
    nsamp = 323 + 2887 + 1
    x = workloads.make_filterbank(cfg, nsamp=nsamp).numpy()
    with _mkplan(a, nsamp=nsamp) as plan:
        assert plan.nout == 1
        _check(plan, x, oracle_mod, 1, exact=True)
    with pytest.raises(gsp.GspError) as ei:
        _mkplan(a, nsamp=nsamp - 1)
    assert ei.value.status == 2


@pytest.mark.parametrize("dtype", ["u8", "f32"])
@pytest.mark.parametrize("nsamp", [70, 130, 300])
def test_inputs_shorter_than_a_tma_box(oracle_mod, dtype, nsamp):
    """Fewer input rows than one TMA box (128 / 256 rows) on shapes that otherwise run the streaming
    kernels: the result is still the oracle's (the library may pick another kernel)."""
    rng = np.random.default_rng(nsamp)
    dms = np.arange(0.0, 2.0, 0.25)
    a = dict(nchan=256, f_top=1500.0, chan_bw=-500.0 / 256, dt=98.304e-6, nsamp=nsamp, nsub=4,
             subband_dm=1.0, dm_list=dms, downsamp=1, dtype=dtype)
    x = (rng.integers(0, 256, size=(nsamp, 256), dtype=np.uint8) if dtype == "u8"
         else rng.integers(-50, 50, size=(nsamp, 256)).astype(np.float32))
    with _mkplan(a) as plan:
        _check(plan, x, oracle_mod, 1, exact=True)


def test_bad_pointers_and_options_rejected():
    cfg = workloads.get_config("tiny")
    a = workloads.plan_args(cfg)
    with _mkplan(a) as plan:
        with pytest.raises(gsp.GspError):
            plan.dedisperse(0, 0)
        x = torch.zeros((8192, 64), dtype=torch.uint8, device="cuda")
        out = torch.zeros((plan.ndm, plan.out_pitch + 1), dtype=torch.float32, device="cuda")
        with pytest.raises(gsp.GspError):
            plan.dedisperse(x.data_ptr() + 1, out)          # misaligned input
        with pytest.raises(gsp.GspError):
            plan.set_impl(3, gsp.GSP_IMPL_AUTO)
        with pytest.raises(gsp.GspError):
            plan.set_impl(2, 7)
    a1 = dict(a, nsub=1)
    with _mkplan(a1) as plan:
        with pytest.raises(gsp.GspError):
            plan.set_impl(2, gsp.GSP_IMPL_TILED)            # unsupported shape
        assert plan.get_impl(2) == gsp.GSP_IMPL_GENERIC


# --------------------------------------------------------------------------- float32
F32_IMPLS = [(gsp.GSP_IMPL_GENERIC, gsp.GSP_IMPL_GENERIC), (gsp.GSP_IMPL_AUTO, gsp.GSP_IMPL_AUTO),
             (gsp.GSP_IMPL_AUTO, gsp.GSP_IMPL_GENERIC), (gsp.GSP_IMPL_GENERIC, gsp.GSP_IMPL_AUTO)]


@pytest.mark.parametrize("impl2", F32_IMPLS, ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
@pytest.mark.parametrize("ds", [1, 2, 4, 8])
def test_float32_within_tolerance(oracle_mod, ds, impl2):
    """512 channels in 64 subbands (8 channels each: generic stage 1 whatever is asked, tiled or
    generic stage 2)."""
    cfg = workloads.get_config("ddplan", nchan=512, chan_bw=-500.0 / 512)
    nsamp = 40000
    dms = np.arange(0, 64, 0.5) + 10.0 * ds
    a = dict(nchan=512, f_top=1500.0, chan_bw=-500.0 / 512, dt=49.152e-6, nsamp=nsamp, nsub=64,
             subband_dm=float(dms.mean()), dm_list=dms, downsamp=ds, dtype="f32")
    x = workloads.make_filterbank(cfg, nsamp=nsamp).numpy()
    with _mkplan(a) as plan:
        plan.set_impl(1, gsp.GSP_IMPL_GENERIC if impl2[0] == gsp.GSP_IMPL_GENERIC else gsp.GSP_IMPL_AUTO)
        plan.set_impl(2, impl2[1])
        _check(plan, x, oracle_mod, ds, exact=False)


@pytest.mark.parametrize("impl2", F32_IMPLS, ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
@pytest.mark.parametrize("case", [
    dict(nchan=1024, nsub=16, ds=1, dm0=0.0, ddm=0.5, ndm=100, nsamp=30011),      # cps 64, 4 passes
    dict(nchan=1024, nsub=32, ds=4, dm0=600.0, ddm=2.0, ndm=70, nsamp=60003),     # wide shift spreads
    dict(nchan=512, nsub=32, ds=8, dm0=1200.0, ddm=5.0, ndm=37, nsamp=90001, tile=True),   # cps 16, spread > ring
    dict(nchan=2048, nsub=64, ds=2, dm0=300.0, ddm=1.0, ndm=130, nsamp=50000),
    dict(nchan=1024, nsub=8, ds=16, dm0=100.0, ddm=3.0, ndm=40, nsamp=70001),     # cps 128: clusters of 8
    dict(nchan=256, nsub=16, ds=1, dm0=0.0, ddm=1.0, ndm=33, nsamp=20000),        # cps 16: clusters of 1
    dict(nchan=512, nsub=8, ds=2, dm0=1500.0, ddm=4.0, ndm=20, nsamp=120000, tile=True),   # spread > ring: tile kernel
], ids=lambda c: f"{c['nchan']}ch_{c['nsub']}sub_ds{c['ds']}")
def test_float32_tiled_kernels_within_tolerance(oracle_mod, case, impl2):
    """Shapes the float32 tiled kernels cover (16 | channels per subband): tiled and generic
    kernels in all four pairings against the binary64 oracle."""
    nchan = case["nchan"]
    cfg = workloads.get_config("ddplan", nchan=nchan, chan_bw=-500.0 / nchan)
    dms = case["dm0"] + case["ddm"] * np.arange(case["ndm"])
    a = dict(nchan=nchan, f_top=1500.0, chan_bw=-500.0 / nchan, dt=49.152e-6, nsamp=case["nsamp"],
             nsub=case["nsub"], subband_dm=float(dms.mean()), dm_list=dms, downsamp=case["ds"], dtype="f32")
    x = workloads.make_filterbank(cfg, nsamp=case["nsamp"]).numpy()
    with _mkplan(a) as plan:
        _set(plan, impl2)
        if impl2 == (gsp.GSP_IMPL_AUTO, gsp.GSP_IMPL_AUTO):
            assert (plan.get_impl(1), plan.get_impl(2)) == (gsp.GSP_IMPL_TILED, gsp.GSP_IMPL_TILED)
            assert plan.stage1_split[4] == (0 if case.get("tile") else 1)
        _check(plan, x, oracle_mod, case["ds"], exact=False)


@pytest.mark.parametrize("impl2", F32_IMPLS, ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
def test_float32_integer_valued_input_is_exact(oracle_mod, impl2):
    """Small integers in float32 sum exactly in any order: every kernel pairing is bit-exact."""
    rng = np.random.default_rng(8)
    a = dict(nchan=128, f_top=1500.0, chan_bw=-3.90625, dt=98.304e-6, nsamp=9000, nsub=8,
             subband_dm=50.0, dm_list=np.arange(0, 100, 4.0), downsamp=2, dtype="f32")
    x = rng.integers(0, 256, size=(9000, 128)).astype(np.float32)
    with _mkplan(a) as plan:
        _set(plan, impl2)
        _check(plan, x, oracle_mod, 2, exact=True)


# --------------------------------------------------------------------------- configs 2, 3 (slices)
@pytest.mark.parametrize("impl2", IMPLS, ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
def test_crafts_like_slice_bit_exact(oracle_mod, impl2):
    """CRAFTS-like plan (4096 ch, 64 subbands, 1024 DMs) on a 2^17-sample slice: spans
    82 time tiles x 32 DM blocks of the tiled kernel, with a ragged last tile."""
    cfg = workloads.get_config("crafts")
    nsamp = (1 << 17) + 77
    a = workloads.plan_args(cfg, nsamp=nsamp)
    x = workloads.make_filterbank(cfg, device="cuda", nsamp=nsamp).cpu().numpy()
    with _mkplan(a) as plan:
        _set(plan, impl2)
        assert (plan.H1, plan.H2) == (656, 46638)
        _check(plan, x, oracle_mod, 1, exact=True)


def test_uwb_like_slice_bit_exact(oracle_mod):
    """UWB-like plan (128 subbands, 512 DMs, downsamp 2, halo 276,342 rows) on 2^19 samples."""
    cfg = workloads.get_config("uwb")
    nsamp = (1 << 19) + 3
    a = workloads.plan_args(cfg, nsamp=nsamp)
    x = workloads.make_filterbank(cfg, device="cuda", nsamp=nsamp).cpu().numpy()
    with _mkplan(a) as plan:
        assert (plan.H1, plan.H2) == (10552, 132895)
        _check(plan, x, oracle_mod, 2, exact=True)


# --------------------------------------------------------------------------- streaming / host path
@pytest.mark.parametrize("ds", [1, 2])
def test_block_carry_streaming_equals_one_shot(oracle_mod, ds):
    """Config-5 semantic at small scale: consecutive blocks with the halo carried give the
    one-shot output (Algorithm 1's lastdata/data)."""
    cfg = workloads.get_config("tiny")
    a = workloads.plan_args(cfg)
    a["downsamp"] = ds
    B, nblk = 8192, 4
    x = workloads.make_filterbank(cfg, nsamp=B * nblk)
    xd = x.cuda()
    with _mkplan(a, nsamp=B * nblk) as full, _mkplan(a, nsamp=B) as first:
        H = full.halo
        y_full = _run(full, xd)
        parts = [_run(first, xd[:B].contiguous())]
        nout0 = first.nout
        with _mkplan(a, nsamp=B + H) as blk:
            assert blk.nout == B // ds
            for k in range(1, nblk):
                start = ds * nout0 + (k - 1) * B
                parts.append(_run(blk, xd[start:start + B + H].contiguous()))
        cat = np.concatenate(parts, axis=1)
        np.testing.assert_array_equal(cat, y_full[:, : cat.shape[1]])
        s1, s2 = _oracle_tables(full, oracle_mod)
        want = oracle_mod.dedisperse(x.numpy(), s1, s2, ds)
        np.testing.assert_array_equal(y_full, want)


@pytest.mark.parametrize("dtype", ["u8", "f32"])
def test_host_buffer_path_equals_device_path(oracle_mod, dtype):
    cfg = workloads.get_config("tiny", dtype=dtype)
    a = workloads.plan_args(cfg)
    nsamp = 300000                       # several internal chunks
    x = workloads.make_filterbank(cfg, nsamp=nsamp)
    with _mkplan(a, nsamp=nsamp) as plan:
        y_dev = _run(plan, x.cuda())
        h_in = x.pin_memory()
        h_out = torch.zeros((plan.ndm, plan.nout), dtype=torch.float32).pin_memory()
        plan.dedisperse_host(h_in, h_out, plan.nout)
        np.testing.assert_array_equal(h_out.numpy(), y_dev)
        if dtype == "u8":
            s1, s2 = _oracle_tables(plan, oracle_mod)
            want = oracle_mod.dedisperse(x.numpy(), s1, s2, 1, nthreads=oracle_mod.max_threads())
            np.testing.assert_array_equal(y_dev, want)


@pytest.mark.parametrize("dtype", ["u8", "f32"])
def test_host_buffer_path_with_streaming_kernels_is_bit_identical(dtype):
    """Chunked host-buffer path against the one-shot device path on a shape that runs the streaming
    stage-1 kernels (TMA rings, clusters) and the tiled stage 2: the summation order of every output
    does not depend on where a chunk starts, so both dtypes agree bit for bit (pin P10)."""
    rng = np.random.default_rng(77)
    nsamp, nchan = 260000, 256
    dms = np.arange(0.0, 40.0, 1.0)
    a = dict(nchan=nchan, f_top=1500.0, chan_bw=-500.0 / nchan, dt=49.152e-6, nsamp=nsamp, nsub=4,
             subband_dm=20.0, dm_list=dms, downsamp=1 if dtype == "u8" else 2, dtype=dtype)
    x = (torch.from_numpy(rng.integers(0, 256, size=(nsamp, nchan), dtype=np.uint8)) if dtype == "u8"
         else torch.from_numpy(rng.standard_normal((nsamp, nchan)).astype(np.float32)))
    with _mkplan(a) as plan:
        assert (plan.get_impl(1), plan.get_impl(2)) == (gsp.GSP_IMPL_TILED, gsp.GSP_IMPL_TILED)
        split = plan.stage1_split
        assert split[0] > 0 if dtype == "u8" else split[4] == 1
        y_dev = _run(plan, x.cuda())
        h_in = x.pin_memory()
        h_out = torch.zeros((plan.ndm, plan.nout), dtype=torch.float32).pin_memory()
        plan.dedisperse_host(h_in, h_out, plan.nout)
        np.testing.assert_array_equal(h_out.numpy(), y_dev)
        # host input, device output: the same chunks gathered on the device, padding columns untouched
        d_out = torch.full((plan.ndm, plan.out_pitch), -12345.0, dtype=torch.float32, device="cuda")
        plan.dedisperse_host_in(h_in, d_out, plan.out_pitch)
        got = d_out.cpu().numpy()
        np.testing.assert_array_equal(got[:, : plan.nout], y_dev)
        assert np.all(got[:, plan.nout:] == -12345.0)
        with pytest.raises(gsp.GspError):
            plan.dedisperse_host_in(h_in, d_out, plan.nout - 1)


@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_dedisperse_multi_equals_separate_calls(oracle_mod, dtype):
    """gsp_dedisperse_multi over four DM ranges with their own subband DM and downsampling (a small
    DDplan): bit-identical to four gsp_dedisperse calls — float32 plans and uint8 plans each share ONE ring
    (input fetched once, a gather per plan) — and every range against the oracle."""
    rng = np.random.default_rng(5)
    nchan, nsamp = 512, 70000
    x = (rng.standard_normal((nsamp, nchan)).astype(np.float32) if dtype == "f32"
         else rng.integers(0, 256, size=(nsamp, nchan), dtype=np.uint8))
    xd = torch.from_numpy(x).cuda()
    ranges = [(0.0, 0.5, 60, 1), (30.0, 1.0, 30, 2), (60.0, 2.0, 30, 4), (120.0, 5.0, 36, 8)]
    if dtype == "u8":      # subband DMs whose stage-1 shifts all fit the 1024-row ring (the last: int32 operands)
        ranges[3] = (90.0, 2.0, 20, 8)
    plans, outs = [], []
    try:
        for lo, step, n, ds in ranges:
            dms = lo + step * np.arange(n)
            plans.append(_mkplan(dict(nchan=nchan, f_top=1500.0, chan_bw=-500.0 / nchan, dt=49.152e-6, nsamp=nsamp,
                                      nsub=16, subband_dm=float(dms.mean()), dm_list=dms, downsamp=ds, dtype=dtype)))
        assert len({p.nout for p in plans}) > 1          # the plans really differ in length
        assert all((p.get_impl(1), p.get_impl(2)) == (gsp.GSP_IMPL_TILED, gsp.GSP_IMPL_TILED) for p in plans)
        if dtype == "f32":
            assert all(p.stage1_split[4] == 1 for p in plans)
        else:
            assert all(p.stage1_split[0] == nchan // 64 for p in plans)     # every group on the shared ring
        sep = [_run(p, xd) for p in plans]
        outs = [torch.full((p.ndm, p.out_pitch), -12345.0, dtype=torch.float32, device="cuda") for p in plans]
        gsp.dedisperse_multi(plans, xd, outs, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        for p, o, ref in zip(plans, outs, sep):
            got = o.cpu().numpy()
            assert np.all(got[:, p.nout:] == -12345.0)
            np.testing.assert_array_equal(got[:, : p.nout], ref)
        for p, got in zip(plans, sep):
            s1, s2 = _oracle_tables(p, oracle_mod)
            want = oracle_mod.dedisperse(x, s1, s2, p.args["downsamp"], nthreads=oracle_mod.max_threads())
            if dtype == "u8":
                np.testing.assert_array_equal(got, want)
            else:
                assert _f32_err(got, want) <= F32_TOL
        with pytest.raises(gsp.GspError):
            gsp.dedisperse_multi([plans[0], plans[0]], xd, outs[:2])      # the same plan twice
    finally:
        for p in plans:
            p.destroy()


def test_reserve_multi_makes_dedisperse_multi_allocation_free_for_any_grouping():
    """gsp_plan_reserve_multi sizes the float32 shared-ring scratch from the plan alone, so after it
    gsp_dedisperse_multi allocates nothing whichever plans are grouped: the device's free memory does not move
    across calls with different groupings, and the results stay bit-identical to separate calls."""
    rng = np.random.default_rng(8)
    nchan, nsamp = 512, 70000
    xd = torch.from_numpy(rng.standard_normal((nsamp, nchan)).astype(np.float32)).cuda()
    ranges = [(0.0, 1.0, 16, 2), (100.0, 2.0, 16, 2), (200.0, 4.0, 16, 8)]
    plans = []
    try:
        for lo, step, n, ds in ranges:
            dms = lo + step * np.arange(n)
            plans.append(_mkplan(dict(nchan=nchan, f_top=1500.0, chan_bw=-500.0 / nchan, dt=49.152e-6, nsamp=nsamp,
                                      nsub=16, subband_dm=float(dms.mean()), dm_list=dms, downsamp=ds, dtype="f32")))
        sep = [_run(p, xd) for p in plans]
        outs = [torch.empty((p.ndm, p.out_pitch), dtype=torch.float32, device="cuda") for p in plans]
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for p in plans:
            p.reserve_multi()
            p.reserve_multi()                                       # idempotent
        free1 = torch.cuda.mem_get_info()[0]
        per_plan = (nchan // 16) * (-(-nsamp // 32768) * 32768) * 4
        assert free0 - free1 >= 3 * per_plan - (8 << 20) and free0 - free1 <= 3 * per_plan + (64 << 20)
        for group in ([0, 1, 2], [0, 1], [1, 2], [2, 0]):
            sel = [plans[i] for i in group]
            # shared ring: one stage-1 launch + one combine for the whole group (fewer launches from 3 plans on)
            assert gsp.dedisperse_multi_launches(sel) == 2 + len(sel)
            torch.cuda.synchronize()
            before = torch.cuda.mem_get_info()[0]                   # (torch's own pool may have grown since free1)
            gsp.dedisperse_multi(sel, xd, [outs[i] for i in group], torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
            assert torch.cuda.mem_get_info()[0] == before, "gsp_dedisperse_multi allocated after the reservation"
            for i in group:
                np.testing.assert_array_equal(outs[i][:, : plans[i].nout].cpu().numpy(), sep[i])
        with _mkplan(dict(nchan=64, f_top=1500.0, chan_bw=-4.0, dt=49.152e-6, nsamp=9000, nsub=8, subband_dm=5.0,
                          dm_list=np.arange(4.0), downsamp=1, dtype="u8")) as u8plan:
            u8plan.reserve_multi()                                  # nothing to reserve for uint8 plans: a no-op
    finally:
        for p in plans:
            p.destroy()


@pytest.mark.parametrize("case", [
    dict(ranges=[(0.0, 0.5, 24, 16), (40.0, 1.0, 20, 32), (80.0, 2.0, 20, 64), (150.0, 4.0, 12, 128)],
         nsamp=90000, stage1_launches=5),                 # folds of 64 / 128: shared ring + one scalar combine per plan
    dict(ranges=[(0.0, 1.0, 20, 1), (200.0, 5.0, 20, 4)], nsamp=70000, stage1_launches=2),   # shared ring + ONE combine
    dict(ranges=[(0.0, 1.0, 16, 2), (100.0, 2.0, 16, 2), (200.0, 4.0, 16, 8)], nsamp=70000, stage1_launches=2),
    dict(ranges=[(0.0, 1.0, 16, 1), (450.0, 10.0, 16, 4)], nsamp=100000, stage1_launches=1),
    # ^ the second plan's shift spread leaves no room for a shared ring: its clusters run beside the first plan's
], ids=["big_downsamp", "two_plans", "three_plans", "spread_too_wide_for_one_ring"])
def test_dedisperse_multi_f32_shared_ring(oracle_mod, case):
    """float32 gsp_dedisperse_multi: the shared-ring stage 1 (plans working lag_p chunks behind the stream head,
    group partial sums combined by a second kernel) is bit-identical to separate gsp_dedisperse calls for any
    number of plans and any DownSamp, and so is the side-by-side launch it falls back to."""
    rng = np.random.default_rng(len(case["ranges"]) + case["nsamp"])
    nchan, nsamp = 512, case["nsamp"]
    x = rng.standard_normal((nsamp, nchan)).astype(np.float32)
    xd = torch.from_numpy(x).cuda()
    plans = []
    try:
        for lo, step, n, ds in case["ranges"]:
            dms = lo + step * np.arange(n)
            plans.append(_mkplan(dict(nchan=nchan, f_top=1500.0, chan_bw=-500.0 / nchan, dt=49.152e-6, nsamp=nsamp,
                                      nsub=16, subband_dm=float(dms.mean()), dm_list=dms, downsamp=ds, dtype="f32")))
        assert all(p.stage1_split[4] == 1 for p in plans)          # every plan streams (the multi launch applies)
        assert gsp.dedisperse_multi_launches(plans) == case["stage1_launches"] + len(plans)   # which path runs
        sep = [_run(p, xd) for p in plans]
        outs = [torch.full((p.ndm, p.out_pitch), -12345.0, dtype=torch.float32, device="cuda") for p in plans]
        for _ in range(2):                                         # twice: the scratch is reused
            gsp.dedisperse_multi(plans, xd, outs, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        for p, o, ref in zip(plans, outs, sep):
            got = o.cpu().numpy()
            assert np.all(got[:, p.nout:] == -12345.0)
            np.testing.assert_array_equal(got[:, : p.nout], ref)
        for p, got in zip(plans, sep):
            s1, s2 = _oracle_tables(p, oracle_mod)
            want = oracle_mod.dedisperse(x, s1, s2, p.args["downsamp"], nthreads=oracle_mod.max_threads())
            assert _f32_err(got, want) <= F32_TOL
    finally:
        for p in plans:
            p.destroy()


@pytest.mark.parametrize("cps", [64, 32, 16])
@pytest.mark.parametrize("ds", [2, 4, 8, 16, 32, 64, 128])
def test_uint8_downsampling_runs_the_product_kernels(oracle_mod, cps, ds):
    """The DownSamp column of the paper's DDplans (Tables 2-3: 1 ... 128): uint8 plans with
    any of those factors run the streaming stage 1 and the TILED stage 2 — packed u16 operands folded every
    4, 2 or 1 subbands while cps*255*ds fits 16 bits, int32 operands beyond — bit-exact."""
    rng = np.random.default_rng(1000 * cps + ds)
    nsub = 8
    nchan = cps * nsub
    dms = 4.0 * ds * (20.0 + np.arange(0.0, 37.0, 1.0))
    a = dict(nchan=nchan, f_top=1500.0, chan_bw=-(300.0 / ds) / nchan, dt=49.152e-6, nsamp=0, nsub=nsub,
             subband_dm=float(dms.mean()), dm_list=dms, downsamp=ds, dtype="u8")
    s1, s2 = oracle_mod.delay_tables(nchan, a["f_top"], a["chan_bw"], a["dt"], nsub, a["subband_dm"], dms, ds)
    assert s1.max() <= 768 and s2.max() >= 20
    nsamp = a["nsamp"] = int(s1.max()) + ds * (int(s2.max()) + 2100 + 1024 // ds) + ds - 1   # ragged tail
    x = rng.integers(0, 256, size=(nsamp, nchan), dtype=np.uint8)
    x[rng.integers(0, nsamp, 50)] = 255                   # saturated rows: the lane bounds are reached
    with _mkplan(a) as plan:
        assert plan.get_impl(2) == gsp.GSP_IMPL_TILED
        assert plan.get_impl(1) == gsp.GSP_IMPL_TILED
        if nchan % 64 == 0:
            assert plan.stage1_split[0] == nchan // 64     # streaming ring kernel, not a fallback
        _check(plan, x, oracle_mod, ds, exact=True)
        assert plan.nout > 300


@pytest.mark.parametrize("impl2", IMPLS[:4], ids=lambda i: f"s1-{i[0]}_s2-{i[1]}")
@pytest.mark.parametrize("ds", [1, 2, 8])
def test_one_stage_plan_runs_the_transposing_stage1_and_tiled_stage2(oracle_mod, impl2, ds):
    """nsub == nchan is Algorithm 2 of the paper: one shift per (DM, channel), no subband
    approximation.  Stage 1 is then a pure transposition (+ downsample) with a kernel of its own, and the
    sum runs on the tiled stage 2 with 256 "subbands"."""
    rng = np.random.default_rng(40 + ds)
    nchan, nsamp = 256, 30000 + 37
    dms = np.arange(0.0, 80.0, 2.0)
    a = dict(nchan=nchan, f_top=1500.0, chan_bw=-1.0, dt=98.304e-6, nsamp=nsamp, nsub=nchan, subband_dm=0.0,
             dm_list=dms, downsamp=ds, dtype="u8")
    x = rng.integers(0, 256, size=(nsamp, nchan), dtype=np.uint8)
    with _mkplan(a) as plan:
        _set(plan, impl2)
        if impl2 == (gsp.GSP_IMPL_AUTO, gsp.GSP_IMPL_AUTO):
            assert (plan.get_impl(1), plan.get_impl(2)) == (gsp.GSP_IMPL_TILED, gsp.GSP_IMPL_TILED)
            assert plan.launches_per_call == 2
        got, want = _check(plan, x, oracle_mod, ds, exact=True)
        assert plan.H1 == 0
    # the one-stage result written out independently: y_d[u] = (1/ds) sum_c sum_k x[(u + s2[d][c]) ds + k][c]
    s2 = _oracle_tables_args(a, oracle_mod)[1]
    d = 17
    ref = np.zeros(want.shape[1], dtype=np.int64)
    for c in range(nchan):
        for k in range(ds):
            ref += x[ds * int(s2[d, c]) + k::ds, c][: want.shape[1]].astype(np.int64)
    np.testing.assert_array_equal(got[d], (ref / ds).astype(np.float32))


def test_plans_created_in_descending_shared_memory_order(oracle_mod):
    """The dynamic shared-memory limit of a kernel instantiation is process-wide: a later plan that needs a
    smaller ring must not lower it for an earlier one (they share stage2_tiled_kernel<DPW, WPL, MODE>)."""
    rng = np.random.default_rng(3)
    nchan, nsamp = 256, 40000
    x = rng.standard_normal((nsamp, nchan)).astype(np.float32)
    xd = torch.from_numpy(x).cuda()
    mk = lambda dms: _mkplan(dict(nchan=nchan, f_top=1500.0, chan_bw=-500.0 / nchan, dt=49.152e-6, nsamp=nsamp,
                                  nsub=16, subband_dm=float(dms.mean()), dm_list=dms, downsamp=1, dtype="f32"))
    big = mk(np.arange(0.0, 128.0, 2.0))            # wide windows: large stages
    small = mk(np.arange(0.0, 16.0, 0.25))          # same (DPW, WPL): small stages
    try:
        assert big.get_impl(2) == small.get_impl(2) == gsp.GSP_IMPL_TILED
        for plan in (small, big, small, big):
            s1, s2 = _oracle_tables(plan, oracle_mod)
            want = oracle_mod.dedisperse(x, s1, s2, 1, nthreads=oracle_mod.max_threads())
            assert _f32_err(_run(plan, xd), want) <= F32_TOL
    finally:
        big.destroy()
        small.destroy()


def test_stage_timing_and_launch_count():
    cfg = workloads.get_config("tiny")
    a = workloads.plan_args(cfg)
    with _mkplan(a) as plan:
        plan.enable_stage_timing(True)
        x = workloads.make_filterbank(cfg).cuda()
        _run(plan, x)
        ms1, ms2 = plan.last_stage_ms()
        assert ms1 > 0 and ms2 > 0
        assert plan.launches_per_call == 2
