"""GPU parity of the RFI prologue (gsp_plan_set_rfi, readings F1-F4 of DESIGN.md §3a) fused into stage 1:
dedispersion of the cleaned filterbank must equal oracle.dedisperse(oracle.rfi_prologue(x)) bit for bit
(uint8: integers everywhere, one binary64 comparison per row), with the streaming ring kernel (prologue
applied to the words entering the shared-memory ring) and with the generic kernel."""
import numpy as np
import pytest
import torch

import paper_2110_12749_b200 as gsp

pytestmark = pytest.mark.gpu


def _input(rng, nsamp, nchan, nburst=25):
    x = rng.normal(128, 12, size=(nsamp, nchan)).round().clip(0, 255).astype(np.uint8)
    for t in rng.integers(0, nsamp, nburst):                       # broadband bursts of a few rows
        w = int(rng.integers(1, 4))
        x[t:t + w] = np.minimum(255, x[t:t + w].astype(int) + int(rng.integers(6, 70))).astype(np.uint8)
    return x


def _run(plan, xd):
    out = torch.full((plan.ndm, plan.out_pitch), -12345.0, dtype=torch.float32, device="cuda")
    plan.dedisperse(xd, out, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out[:, : plan.nout].cpu().numpy()


@pytest.mark.parametrize("impl1", [gsp.GSP_IMPL_AUTO, gsp.GSP_IMPL_GENERIC], ids=["ring", "generic"])
@pytest.mark.parametrize("case", [
    dict(mask=True, sigma=0.0, block=0, ds=1),
    dict(mask=False, sigma=3.0, block=1024, ds=1),
    dict(mask=True, sigma=2.5, block=512, ds=2),
    dict(mask=True, sigma=4.0, block=2048, ds=4),
], ids=["mask", "clip", "mask+clip_ds2", "mask+clip_ds4"])
def test_rfi_prologue_bit_exact(oracle_mod, impl1, case):
    rng = np.random.default_rng(17)
    nchan, nsub, nsamp, ds = 512, 8, 41003, case["ds"]      # ragged last clip block, ragged ring chunks
    dms = np.arange(0.0, 60.0, 1.5)
    a = dict(nchan=nchan, f_top=1500.0, chan_bw=-400.0 / nchan, dt=49.152e-6, nsub=nsub, subband_dm=30.0)
    x = _input(rng, nsamp, nchan)
    mask = (rng.random(nchan) < 0.08).astype(np.uint8) if case["mask"] else None
    pad = rng.integers(110, 150, size=nchan, dtype=np.uint8)
    x2, z, clipped = oracle_mod.rfi_prologue(x, mask, pad, case["sigma"], case["block"])
    if case["sigma"] > 0:
        assert 5 <= clipped.sum() <= 400
    s1, s2 = oracle_mod.delay_tables(nchan, a["f_top"], a["chan_bw"], a["dt"], nsub, a["subband_dm"], dms, ds)
    want = oracle_mod.dedisperse(x2, s1, s2, ds, nthreads=oracle_mod.max_threads())
    with gsp.Plan(nchan, a["f_top"], a["chan_bw"], a["dt"], nsamp, nsub, a["subband_dm"], dms, ds, "u8") as plan:
        plan.set_impl(1, impl1)
        xd = torch.from_numpy(x).cuda()
        plain = _run(plan, xd)
        plan.set_rfi(mask, pad, case["sigma"], case["block"])
        if impl1 == gsp.GSP_IMPL_AUTO:
            assert plan.get_impl(1) == gsp.GSP_IMPL_TILED and plan.stage1_split[0] == nchan // 64
        got = _run(plan, xd)
        assert np.array_equal(got, want), f"{int((got != want).sum())} outputs differ"
        assert not np.array_equal(got, plain)                   # the prologue really changed something
        if case["sigma"] > 0:
            gz, gc = plan.rfi_last()
            np.testing.assert_array_equal(gz, z)
            np.testing.assert_array_equal(gc, clipped)
            assert plan.launches_per_call == 3
        plan.set_rfi(None, None)                                # cleared: back to the plain result
        np.testing.assert_array_equal(_run(plan, xd), plain)


@pytest.mark.parametrize("case", [
    dict(nchan=256, nsub=8, sdm=60.0, ds=1),     # cps 32: common-stream and per-slice long rings, two and one CTA per SM
    dict(nchan=256, nsub=8, sdm=30.0, ds=2),     # cps 32: standard ring + long rings in one plan
    dict(nchan=128, nsub=8, sdm=90.0, ds=4),     # cps 16
    dict(nchan=256, nsub=4, sdm=25.0, ds=1),     # cps 64: four slices, per-slice streams
], ids=lambda c: f"{c['nchan']}ch_{c['nsub']}sub_sdm{c['sdm']:g}")
def test_rfi_prologue_in_the_long_ring_kernels(oracle_mod, case):
    """Low band, wide stage-1 shifts: the prologue (channel mask + zero-DM clip) is applied on the way into the long
    rings as well — common stream and per-slice streams, whose rows start at each slice's own first row — bit-exact
    against oracle.rfi_prologue + oracle.dedisperse."""
    rng = np.random.default_rng(case["nchan"] + int(case["sdm"]))
    nchan, nsub, ds, nsamp = case["nchan"], case["nsub"], case["ds"], 45001
    dms = np.arange(0.0, 12.0, 1.0) * ds
    x = _input(rng, nsamp, nchan)
    mask = (rng.random(nchan) < 0.08).astype(np.uint8)
    pad = rng.integers(110, 150, size=nchan, dtype=np.uint8)
    x2, z, clipped = oracle_mod.rfi_prologue(x, mask, pad, 3.0, 1024)
    assert clipped.sum() >= 5
    s1, s2 = oracle_mod.delay_tables(nchan, 400.0, -128.0 / nchan, 98.304e-6, nsub, case["sdm"], dms, ds)
    want = oracle_mod.dedisperse(x2, s1, s2, ds, nthreads=oracle_mod.max_threads())
    with gsp.Plan(nchan, 400.0, -128.0 / nchan, 98.304e-6, nsamp, nsub, case["sdm"], dms, ds, "u8") as plan:
        split = plan.stage1_split
        assert split[5] + split[6] > 0 and split[1] + split[2] + split[3] == 0, split    # long rings, nothing else
        xd = torch.from_numpy(x).cuda()
        plain = _run(plan, xd)
        plan.set_rfi(mask, pad, 3.0, 1024)
        assert plan.get_impl(1) == gsp.GSP_IMPL_TILED              # the product kernels carry the prologue
        got = _run(plan, xd)
        assert np.array_equal(got, want), f"{int((got != want).sum())} outputs differ"
        assert not np.array_equal(got, plain)
        gz, gc = plan.rfi_last()
        np.testing.assert_array_equal(gz, z)
        np.testing.assert_array_equal(gc, clipped)
        plan.set_rfi(None, None)
        np.testing.assert_array_equal(_run(plan, xd), plain)


def test_rfi_keeps_the_ring_groups_and_runs_only_the_rest_on_the_generic_kernel(oracle_mod):
    """Low band, wide stage-1 shifts: some 64-channel groups leave the ring kernels for the wide / windowed ones,
    which carry no prologue.  With a prologue those subbands — and only those — run the generic kernel (one extra
    launch); the plan stays on the product kernels for the rest.  Both workspace formats (packed u16 for the
    tiled stage 2, int32 for the generic stage 2)."""
    rng = np.random.default_rng(19)
    nchan, nsub, nsamp = 256, 8, 45000
    dms = np.arange(0.0, 12.0, 1.0)
    x = _input(rng, nsamp, nchan)
    mask = np.zeros(nchan, np.uint8)
    mask[[3, 77, 200]] = 1
    pad = np.full(nchan, 128, np.uint8)
    x2, _, clipped = oracle_mod.rfi_prologue(x, mask, pad, 3.0, 1024)
    s1, s2 = oracle_mod.delay_tables(nchan, 400.0, -0.5, 98.304e-6, nsub, 250.0, dms, 1)
    want = oracle_mod.dedisperse(x2, s1, s2, 1, nthreads=oracle_mod.max_threads())
    with gsp.Plan(nchan, 400.0, -0.5, 98.304e-6, nsamp, nsub, 250.0, dms, 1, "u8") as plan:
        ring, mid, big, win, _, lmid, lbig = plan.stage1_split
        assert plan.get_impl(1) == gsp.GSP_IMPL_TILED and ring < nchan // 64
        assert mid + big + win > 0 and ring + lmid + lbig > 0, plan.stage1_split   # a real mix
        xd = torch.from_numpy(x).cuda()
        plan.set_rfi(mask, pad, 3.0, 1024)
        assert plan.get_impl(1) == gsp.GSP_IMPL_TILED              # no longer dropped to the generic stage 1
        # launches: clip statistics + ring / long-ring launches + ONE generic launch for the rest + stage 2
        # (counts[5] lumps the two two-CTA-per-SM long-ring launches together: one or two launches)
        lo = 1 + (ring > 0) + (lmid > 0) + (lbig > 0) + 1 + 1
        assert lo <= plan.launches_per_call <= lo + (lmid > 0)
        np.testing.assert_array_equal(_run(plan, xd), want)
        plan.set_impl(2, gsp.GSP_IMPL_GENERIC)                     # int32 workspace
        np.testing.assert_array_equal(_run(plan, xd), want)
        plan.set_impl(2, gsp.GSP_IMPL_AUTO)
        plan.set_impl(1, gsp.GSP_IMPL_TILED)                       # forcing the product kernels is accepted too
        np.testing.assert_array_equal(_run(plan, xd), want)
        with pytest.raises(gsp.GspError):
            plan.set_impl(1, gsp.GSP_IMPL_WINDOWED)
        plan.set_impl(1, gsp.GSP_IMPL_GENERIC)
        np.testing.assert_array_equal(_run(plan, xd), want)


def test_rfi_runs_the_whole_stage1_on_the_generic_kernel_when_no_ring_kernel_fits(oracle_mod):
    """8 channels per subband: none of the ring kernels takes the plan, so the prologue runs in the generic
    stage 1 for every subband (documented in gsp.h as the slow case)."""
    rng = np.random.default_rng(23)
    nchan, nsub, nsamp = 64, 8, 20000
    dms = np.arange(0.0, 40.0, 4.0)
    x = _input(rng, nsamp, nchan)
    mask = (rng.random(nchan) < 0.1).astype(np.uint8)
    pad = np.full(nchan, 127, np.uint8)
    x2, _, _ = oracle_mod.rfi_prologue(x, mask, pad, 3.0, 512)
    s1, s2 = oracle_mod.delay_tables(nchan, 1500.0, -4.0, 98.304e-6, nsub, 20.0, dms, 1)
    want = oracle_mod.dedisperse(x2, s1, s2, 1, nthreads=oracle_mod.max_threads())
    with gsp.Plan(nchan, 1500.0, -4.0, 98.304e-6, nsamp, nsub, 20.0, dms, 1, "u8") as plan:
        plan.set_rfi(mask, pad, 3.0, 512)
        assert plan.get_impl(1) == gsp.GSP_IMPL_GENERIC
        np.testing.assert_array_equal(_run(plan, torch.from_numpy(x).cuda()), want)
        with pytest.raises(gsp.GspError):
            plan.set_impl(1, gsp.GSP_IMPL_TILED)


def test_rfi_argument_checks():
    dms = np.arange(0.0, 8.0)
    pad = np.zeros(4096, np.uint8)
    with gsp.Plan(4096, 1500.0, -0.1220703125, 49.152e-6, 20000, 64, 4.0, dms, 1, "u8") as plan:
        for sigma, block in ((3.0, 4096), (3.0, 100), (3.0, 16), (-1.0, 1024), (float("nan"), 1024)):
            with pytest.raises(gsp.GspError):
                plan.set_rfi(None, pad, sigma, block)           # 4096*4096*255 >= 2^31; not a multiple of 32; ...
        plan.set_rfi(None, pad, 3.0, 2048)
        h_in = torch.zeros((20000, 4096), dtype=torch.uint8).pin_memory()
        h_out = torch.zeros((plan.ndm, plan.nout), dtype=torch.float32).pin_memory()
        with pytest.raises(gsp.GspError):
            plan.dedisperse_host(h_in, h_out)                   # clip blocks are defined on the whole input
    with gsp.Plan(256, 1500.0, -1.0, 49.152e-6, 20000, 16, 4.0, dms, 1, "f32") as plan:
        with pytest.raises(gsp.GspError):
            plan.set_rfi(None, np.zeros(256, np.uint8), 0.0, 0)  # uint8 plans only
