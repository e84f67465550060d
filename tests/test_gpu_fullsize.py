"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The oracle cannot produce 10^9 outputs in seconds, so these tests compare SAMPLED outputs:
every sampled y_d[u] is computed one by one, straight from the definition, by
`oracle.points` (O4-O6 of SURVEY.md §8(c)).  To keep host memory bounded the oracle is given
time slabs of the input: outputs u in [ua, ub) depend only on input rows
[ua*ds, ub*ds + halo), and by time-shift equivariance (pin P5) the slab's output index is
u - ua.  Slabs sit at the start, at the end (ragged last tile) and across interior tile
boundaries; sampled DMs include the first and last trial and every kind of DM block.

uint8: bit-exact.  float32: |g - r| <= 1e-5 * max(|r|, rms of the sampled oracle row values)
(reading A13 of DESIGN.md §3 with the row rms estimated from the samples).
"""
import numpy as np
import pytest
import torch

import paper_2110_12749_b200 as gsp
import workloads

pytestmark = pytest.mark.gpu

F32_TOL = 1e-5
SLAB_OUT = 1536          # outputs per slab and DM
N_DM = 48                # sampled DMs per slab
N_U = 40                 # sampled outputs per DM and slab


def _mkplan(a, nsamp=None):
    plan = gsp.Plan(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], int(a["nsamp"] if nsamp is None else nsamp),
                    a["nsub"], a["subband_dm"], a["dm_list"], a["downsamp"], a["dtype"])
    plan.args = a
    return plan


def _oracle_tables(plan, oracle_mod):
    """The ORACLE's tables for the plan's arguments (asserted equal to the library's, entry for entry):
    the oracle is never fed the library's own tables."""
    a = plan.args
    s1, s2 = oracle_mod.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"], a["subband_dm"],
                                     a["dm_list"], a["downsamp"])
    np.testing.assert_array_equal(plan.stage1_shifts, s1)
    np.testing.assert_array_equal(plan.stage2_shifts, s2)
    return s1, s2


def _slab_starts(nout, rng, tile=1024):
    """First outputs of the slabs: start, end, and two interior ones straddling tile boundaries."""
    last = max(0, nout - SLAB_OUT)
    mids = [int(rng.integers(1, max(2, nout // tile - 2))) * tile - SLAB_OUT // 2 for _ in range(2)]
    return sorted({0, last, *[min(max(0, m), last) for m in mids]})


def _check_sampled(oracle_mod, x_dev, y_dev, s1, s2, ds, halo, nout, exact, rng, u_offset=0, what=""):
    """Compare y_dev[d, u_offset + u] with the oracle on sampled (d, u) of several time slabs.
    x_dev row 0 is the first input row of output u = 0."""
    ndm = s2.shape[0]
    nbad, nchk, worst = 0, 0, 0.0
    for ua in _slab_starts(nout, rng):
        ub = min(nout, ua + SLAB_OUT)
        rows = slice(ua * ds, ub * ds + halo)
        assert rows.stop <= x_dev.shape[0]
        x_slab = x_dev[rows].cpu().numpy()
        dsel = np.unique(np.concatenate([[0, ndm - 1, ndm // 2], rng.integers(0, ndm, N_DM)]))
        usel = np.unique(np.concatenate([[0, ub - ua - 1], rng.integers(0, ub - ua, N_U)]))
        dd, uu = np.meshgrid(dsel, usel, indexing="ij")
        want = oracle_mod.points(x_slab, s1, s2, ds, dd.ravel(), uu.ravel()).reshape(dd.shape)
        di = torch.from_numpy(dd.ravel()).cuda()
        ui = torch.from_numpy(uu.ravel() + ua + u_offset).cuda()
        got = y_dev[di, ui].cpu().numpy().reshape(dd.shape)
        nchk += got.size
        if exact:
            nbad += int((got != want).sum())
        else:
            rms = np.sqrt((want.astype(np.float64) ** 2).mean(axis=1, keepdims=True))
            den = np.maximum(np.abs(want), rms)
            den[den == 0] = 1.0
            worst = max(worst, float((np.abs(got.astype(np.float64) - want) / den).max()))
    if exact:
        assert nbad == 0, f"{what}: {nbad} of {nchk} sampled outputs differ from the oracle"
    else:
        assert worst <= F32_TOL, f"{what}: max normalised error {worst:.3e} over {nchk} samples"
    return nchk


def _run_full(plan, x):
    y = torch.full((plan.ndm, plan.out_pitch), -12345.0, dtype=torch.float32, device="cuda")
    plan.dedisperse(x, y, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    if plan.out_pitch > plan.nout:
        assert bool((y[:, plan.nout:] == -12345.0).all()), "padding columns must not be written"
    return y


# --------------------------------------------------------------------------- config 2 (bench workload)
def test_crafts_like_full_size_sampled(oracle_mod):
    """BASELINE configs[1] at full size (2^20 x 4096 uint8, 1024 DMs), default (tiled) kernels =
    exactly what bench.py times."""
    cfg = workloads.get_config("crafts")
    a = workloads.plan_args(cfg)
    rng = np.random.default_rng(20)
    x = workloads.make_filterbank(cfg, device="cuda")
    with _mkplan(a) as plan:
        assert (plan.get_impl(1), plan.get_impl(2)) == (gsp.GSP_IMPL_TILED, gsp.GSP_IMPL_TILED)
        assert plan.nout == 1001282
        y = _run_full(plan, x)
        s1, s2 = _oracle_tables(plan, oracle_mod)
        n = _check_sampled(oracle_mod, x, y, s1, s2, 1, plan.halo, plan.nout, True, rng, what="crafts")
        assert n > 5000
        # the injected pulses are there (E4 of the paper): boxcar S/N at the nearest
        # trial DM and the injected arrival sample, window = pulse width + intra-subband smear
        best = 0.0
        for pu in workloads.pulse_table(cfg):
            if pu["t0"] + 2048 >= plan.nout:
                continue
            d = int(round(pu["dm"]))
            W = int(pu["width"] + abs(pu["dm"] - a["subband_dm"]) * plan.H1 / a["subband_dm"]) + 1
            row = y[d, : plan.nout]
            z = float((row[pu["t0"]: pu["t0"] + W].sum() - W * row.mean()) / (row.std() * W ** 0.5))
            best = max(best, z)
        assert best > 6.0, f"brightest injected pulse only {best:.1f} sigma"


def test_crafts_like_full_size_every_output(oracle_mod):
    """BASELINE configs[1], the bench workload, in the launch configuration bench.py times: ALL
    1024 x 1,001,282 outputs against oracle.dedisperse, element by element ("the GPU results
    are the same as CPU"; one oracle pass over the beam on the box's host cores)."""
    cfg = workloads.get_config("crafts")
    a = workloads.plan_args(cfg)
    x = workloads.make_filterbank(cfg, device="cuda")
    with _mkplan(a) as plan:
        assert (plan.get_impl(1), plan.get_impl(2)) == (gsp.GSP_IMPL_TILED, gsp.GSP_IMPL_TILED)
        y = _run_full(plan, x)
        s1, s2 = _oracle_tables(plan, oracle_mod)
        want = oracle_mod.dedisperse(x.cpu().numpy(), s1, s2, 1, nthreads=oracle_mod.max_threads())
        assert want.shape == (plan.ndm, plan.nout)
        nbad = 0
        for d0 in range(0, plan.ndm, 128):               # compare in slabs of DM rows (bounded host memory)
            got = y[d0:d0 + 128, : plan.nout].cpu().numpy()
            nbad += int((got != want[d0:d0 + 128]).sum())
        assert nbad == 0, f"{nbad} of {want.size} outputs differ from the oracle"


# --------------------------------------------------------------------------- config 3
def test_uwb_like_full_size_sampled(oracle_mod):
    """BASELINE configs[2] at full size (2^21 x 4096 uint8, 128 subbands, 512 DMs, downsamp 2,
    halo 276,342 rows)."""
    cfg = workloads.get_config("uwb")
    a = workloads.plan_args(cfg)
    rng = np.random.default_rng(21)
    x = workloads.make_filterbank(cfg, device="cuda")
    with _mkplan(a) as plan:
        assert (plan.nout, plan.halo) == (910405, 276342)
        y = _run_full(plan, x)
        s1, s2 = _oracle_tables(plan, oracle_mod)
        _check_sampled(oracle_mod, x, y, s1, s2, 2, plan.halo, plan.nout, True, rng, what="uwb")


def _assert_every_output(y, want, nout, what):
    """y (device, [ndm][pitch]) against the oracle's full result, in slabs of DM rows (bounded host memory)."""
    nbad = 0
    for d0 in range(0, want.shape[0], 128):
        got = y[d0:d0 + 128, :nout].cpu().numpy()
        nbad += int((got != want[d0:d0 + 128]).sum())
    assert nbad == 0, f"{what}: {nbad} of {want.size} outputs differ from the oracle"


def test_uwb_like_full_size_every_output(oracle_mod):
    """BASELINE configs[2] at full size on EVERY output (512 x 910,405): the ring kernel and both long-ring
    launches of stage 1, DownSamp 2, every DM block x time tile of stage 2 including the once-per-plan corners
    a sampled comparison can miss (one oracle pass over the 8 GiB beam on the host cores)."""
    cfg = workloads.get_config("uwb")
    a = workloads.plan_args(cfg)
    x = workloads.make_filterbank(cfg, device="cuda")
    with _mkplan(a) as plan:
        assert (plan.get_impl(1), plan.get_impl(2)) == (gsp.GSP_IMPL_TILED, gsp.GSP_IMPL_TILED)
        split = plan.stage1_split
        assert split[0] > 0 and split[5] > 0 and split[6] > 0, split       # ring + both kinds of long ring
        y = _run_full(plan, x)
        s1, s2 = _oracle_tables(plan, oracle_mod)
        want = oracle_mod.dedisperse(x.cpu().numpy(), s1, s2, 2, nthreads=oracle_mod.max_threads())
        assert want.shape == (plan.ndm, plan.nout)
        _assert_every_output(y, want, plan.nout, "uwb")


def test_paper_band1_ddplan_full_size_every_output(oracle_mod):
    """Table 2 of the paper on the Band1 shape: all 8 ranges (3462 DMs, DownSamp 1 ... 128) in one
    gsp_dedisperse_multi call, EVERY output of every range against oracle.dedisperse."""
    cfg = workloads.get_config("band1")
    x = workloads.make_filterbank(cfg, device="cuda")
    x_np = x.cpu().numpy()
    plans = []
    try:
        for pi in range(len(cfg["plans"])):
            plans.append(_mkplan(workloads.plan_args(cfg, pi)))
        outs = [torch.full((p.ndm, p.out_pitch), -12345.0, dtype=torch.float32, device="cuda") for p in plans]
        gsp.dedisperse_multi(plans, x, outs, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        total = 0
        for pi, (p, y) in enumerate(zip(plans, outs)):
            s1, s2 = _oracle_tables(p, oracle_mod)
            want = oracle_mod.dedisperse(x_np, s1, s2, p.args["downsamp"], nthreads=oracle_mod.max_threads())
            assert want.shape == (p.ndm, p.nout)
            _assert_every_output(y, want, p.nout, f"band1 range {pi}")
            total += want.size
        assert total > 5e8
    finally:
        for p in plans:
            p.destroy()


# --------------------------------------------------------------------------- config 4
def test_ddplan_float32_full_size_sampled(oracle_mod):
    """BASELINE configs[3]: 2^21 x 4096 float32 (32 GiB), four DM ranges back to back with
    downsamp 1/2/4/8, each against the binary64 oracle at 1e-5."""
    cfg = workloads.get_config("ddplan")
    free, _ = torch.cuda.mem_get_info()
    if free < 60 * 2**30:
        pytest.skip("needs 60 GiB of free device memory")
    rng = np.random.default_rng(22)
    x = workloads.make_filterbank(cfg, device="cuda")
    want_nout = [2083306, 1034633, 510345, 244739]
    plans, ys = [], []
    try:
        for pi in range(len(cfg["plans"])):
            a = workloads.plan_args(cfg, pi)
            plan = _mkplan(a)
            plans.append(plan)
            assert plan.nout == want_nout[pi]
            assert plan.stage1_split[4] == 1                   # the streaming stage-1 kernel runs every range
            y = _run_full(plan, x)
            s1, s2 = _oracle_tables(plan, oracle_mod)
            _check_sampled(oracle_mod, x, y, s1, s2, a["downsamp"], plan.halo, plan.nout, False, rng,
                           what=f"ddplan range {pi}")
            ys.append(y)
        # the four ranges "back to back" in one gsp_dedisperse_multi call (shared stage-1 launch):
        # bit-identical to the separate calls
        outs = [torch.full_like(y, -12345.0) for y in ys]
        gsp.dedisperse_multi(plans, x, outs, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        for pi, (y, o) in enumerate(zip(ys, outs)):
            assert torch.equal(y, o), f"ddplan range {pi}: gsp_dedisperse_multi differs from gsp_dedisperse"
    finally:
        for plan in plans:
            plan.destroy()


# --------------------------------------------------------------------------- the paper's own DDplans
@pytest.mark.parametrize("band", ["band1", "band2"])
def test_paper_ddplans_full_size_sampled(oracle_mod, band):
    """Tables 2 and 3 of the paper on the Band1 / Band2 shapes of Table 1:
    8 ranges / 3462 DMs on 512 channels, 6 ranges / 10,730 DMs on 2048 channels, DownSamp 1 ... 128, uint8,
    all ranges in one gsp_dedisperse_multi call (shared stage-1 ring where the ranges allow); sampled outputs
    of every range against the oracle, and the call bit-identical to separate gsp_dedisperse calls."""
    cfg = workloads.get_config(band)
    rng = np.random.default_rng(31)
    x = workloads.make_filterbank(cfg, device="cuda")
    plans, outs = [], []
    try:
        for pi in range(len(cfg["plans"])):
            plans.append(_mkplan(workloads.plan_args(cfg, pi)))
        assert sum(p.ndm for p in plans) == {"band1": 3462, "band2": 10730}[band]
        assert all(p.get_impl(2) == gsp.GSP_IMPL_TILED for p in plans)      # every DownSamp on the product stage 2
        assert all(p.get_impl(1) == gsp.GSP_IMPL_TILED for p in plans)
        outs = [torch.full((p.ndm, p.out_pitch), -12345.0, dtype=torch.float32, device="cuda") for p in plans]
        gsp.dedisperse_multi(plans, x, outs, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        for pi, (p, y) in enumerate(zip(plans, outs)):
            if p.out_pitch > p.nout:
                assert bool((y[:, p.nout:] == -12345.0).all())
            s1, s2 = _oracle_tables(p, oracle_mod)
            _check_sampled(oracle_mod, x, y, s1, s2, p.args["downsamp"], p.halo, p.nout, True, rng,
                           what=f"{band} range {pi}")
            assert torch.equal(_run_full(p, x), y), f"{band} range {pi}: multi differs from a separate call"
    finally:
        for p in plans:
            p.destroy()


# --------------------------------------------------------------------------- config 5
@pytest.mark.parametrize("beam", [0, 18])
def test_stream19_beam_in_blocks_full_size_sampled(oracle_mod, beam):
    """BASELINE configs[4], one beam at full size: 2^21 samples dedispersed as 4 consecutive
    blocks of 2^19 with the halo carried (first block: plan of B rows; later blocks: plan of
    B + H rows emitting exactly B outputs), concatenated output against the oracle."""
    cfg = workloads.get_config("stream19")
    a = workloads.plan_args(cfg)
    B, nblk = cfg["block"], cfg["nblocks"]
    rng = np.random.default_rng(23 + beam)
    x = workloads.make_filterbank(cfg, device="cuda", seed=cfg["seed"] + beam)
    assert x.shape[0] == B * nblk
    stream = torch.cuda.current_stream().cuda_stream
    with _mkplan(a, nsamp=B) as first:
        H = first.halo
        assert H == 47294
        with _mkplan(a, nsamp=B + H) as blk:
            assert blk.nout == B
            nout_total = first.nout + (nblk - 1) * B
            y = torch.empty((first.ndm, nout_total), dtype=torch.float32, device="cuda")
            tmp0 = torch.empty((first.ndm, first.out_pitch), dtype=torch.float32, device="cuda")
            first.dedisperse(x[:B], tmp0, stream)
            y[:, : first.nout] = tmp0[:, : first.nout]
            tmp = torch.empty((blk.ndm, blk.out_pitch), dtype=torch.float32, device="cuda")
            for k in range(1, nblk):
                start = first.nout + (k - 1) * B            # first output of block k == its first input row
                blk.dedisperse(x[start:start + B + H], tmp, stream)
                y[:, start:start + B] = tmp[:, :B]
            torch.cuda.synchronize()
            s1, s2 = _oracle_tables(first, oracle_mod)
            np.testing.assert_array_equal(blk.stage1_shifts, s1)
            np.testing.assert_array_equal(blk.stage2_shifts, s2)
            _check_sampled(oracle_mod, x, y, s1, s2, 1, H, nout_total, True, rng, what=f"stream19 beam {beam}")
