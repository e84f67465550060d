"""GPU parity of the single-pulse search (gsp_search_*, through the C ABI) against the oracle's
`search` (readings S1-S6).  Every float decision is taken in a stated precision and
order, so there is exactly one result: the candidate list (DM, sample, width: integers) must be
bit-exact, and so must the float32 snr and the block statistics.
"""
import numpy as np
import pytest
import torch

import paper_2110_12749_b200 as gsp
import workloads

pytestmark = pytest.mark.gpu


def _gpu_search(y_dev, nout, block, nwidths, thr, max_cand=None, want_stats=True):
    ndm, pitch = y_dev.shape
    with gsp.Search(ndm, nout, pitch, block, nwidths, thr, ndm * ((nout + block - 1) // block)
                    if max_cand is None else max_cand) as s:
        cap = max(1, s.max_cand)
        dm = torch.full((cap,), -7, dtype=torch.int32, device="cuda")
        u = torch.full((cap,), -7, dtype=torch.int32, device="cuda")
        w = torch.full((cap,), -7, dtype=torch.int32, device="cuda")
        snr = torch.full((cap,), -7.0, dtype=torch.float32, device="cuda")
        cnt = torch.zeros((1,), dtype=torch.int64, device="cuda")
        stats = torch.zeros((ndm, s.nblocks, 2), dtype=torch.float32, device="cuda") if want_stats else None
        s.run(y_dev, dm, u, w, snr, cnt, stats, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        n = int(cnt.item())
        k = min(n, s.max_cand)
        assert bool((dm[k:] == -7).all()) or s.max_cand == 0, "entries past the count must not be written"
        return dict(count=n, dm=dm[:k].cpu().numpy(), sample=u[:k].cpu().numpy(), width=w[:k].cpu().numpy(),
                    snr=snr[:k].cpu().numpy(), stats=None if stats is None else stats.cpu().numpy())


def _same(got, want, stats=True):
    assert got["count"] == want["count"]
    np.testing.assert_array_equal(got["dm"], want["dm"])
    np.testing.assert_array_equal(got["sample"], want["sample"])
    np.testing.assert_array_equal(got["width"], want["width"])
    np.testing.assert_array_equal(got["snr"], want["snr"])
    if stats:
        np.testing.assert_array_equal(got["stats"], want["stats"])


@pytest.mark.parametrize("block", [256, 512, 1024, 2048])
@pytest.mark.parametrize("nwidths", [1, 3, 4, 5, 6])
def test_search_noise_every_block_bit_exact(oracle_mod, block, nwidths):
    """threshold = -inf-ish: every (DM, block) reports its winner — the whole argmax machinery, the ragged last
    block, rows whose pitch exceeds nout (garbage past nout must be ignored), several runs of blocks per row."""
    rng = np.random.default_rng(block + nwidths)
    ndm, nout, pitch = 5, 19 * block + 333, 19 * block + 352
    y = (rng.normal(0, 40, size=(ndm, pitch)) + 524288.0).round().astype(np.float32)
    y[:, nout:] = np.float32(9e9)                          # padding columns: never read as data
    want = oracle_mod.search(y, nout=nout, block=block, nwidths=nwidths, threshold=-1e30, return_stats=True)
    got = _gpu_search(torch.from_numpy(y).cuda(), nout, block, nwidths, -1e30)
    assert want["count"] == ndm * (-(-nout // block))
    _same(got, want)


def test_search_non_integer_float_input_bit_exact(oracle_mod):
    """float32 series that are not integers (the float32 dedispersion path): the tree order makes the
    binary64 sums — and everything after them — reproducible bit for bit."""
    rng = np.random.default_rng(3)
    ndm, nout = 7, 40000
    y = rng.normal(0.3, 8.0, size=(ndm, nout)).astype(np.float32)
    for d in range(ndm):
        y[d, 3000 + 5000 * d: 3000 + 5000 * d + (1 << (d % 6))] += 30.0
    want = oracle_mod.search(y, block=1024, nwidths=6, threshold=-1e30, return_stats=True)
    got = _gpu_search(torch.from_numpy(y).cuda(), nout, 1024, 6, -1e30)
    _same(got, want)


def test_search_threshold_compaction_capacity_and_order(oracle_mod):
    rng = np.random.default_rng(4)
    ndm, nout = 300, 30000
    y = rng.normal(0, 1, size=(ndm, nout)).astype(np.float32)
    yd = torch.from_numpy(y).cuda()
    want = oracle_mod.search(y, block=512, nwidths=6, threshold=3.5)
    assert 50 < want["count"] < ndm * 59
    _same(_gpu_search(yd, nout, 512, 6, 3.5, want_stats=False), want, stats=False)
    cap = oracle_mod.search(y, block=512, nwidths=6, threshold=3.5, max_cand=17)
    got = _gpu_search(yd, nout, 512, 6, 3.5, max_cand=17, want_stats=False)
    _same(got, cap, stats=False)
    assert got["count"] == want["count"] and len(got["dm"]) == 17
    none = _gpu_search(yd, nout, 512, 6, 50.0, want_stats=False)
    assert none["count"] == 0
    cnt_only = _gpu_search(yd, nout, 512, 6, 3.5, max_cand=0, want_stats=False)
    assert cnt_only["count"] == want["count"]


def test_search_degenerate_inputs(oracle_mod):
    y = np.full((3, 5000), 524288.0, dtype=np.float32)     # constant: var = 0, no candidate
    assert _gpu_search(torch.from_numpy(y).cuda(), 5000, 1024, 6, 1e-3)["count"] == 0
    for thr in (0.0, -1.0):                                # ... but it IS one for threshold <= 0 (gsp.h): snr 0, width 1
        got = _gpu_search(torch.from_numpy(y).cuda(), 5000, 1024, 6, thr)
        _same(got, oracle_mod.search(y, block=1024, nwidths=6, threshold=thr, return_stats=True))
        assert got["count"] == 15 and np.all(got["snr"] == 0.0) and np.all(got["width"] == 1)
    y = np.full((2, 2048), 7.0, dtype=np.float32)          # constant block, then a pulse right behind its end:
    y[:, 1024:] = 0.0                                      # a boxcar starting in the constant block reaches it
    y[:, 1024:1026] = 100.0
    got = _gpu_search(torch.from_numpy(y).cuda(), 2048, 1024, 6, 5.0)
    _same(got, oracle_mod.search(y, block=1024, nwidths=6, threshold=5.0, return_stats=True))
    assert got["count"] == 4 and (int(got["sample"][0]), int(got["width"][0])) == (1022, 4)
    y = np.zeros((1, 1024), dtype=np.float32)              # exact tie between two widths (oracle pin)
    y[0, 200:204] = 1025.0
    y[0, 600] = 2044.0
    got = _gpu_search(torch.from_numpy(y).cuda(), 1024, 1024, 3, 1.0)
    assert (int(got["sample"][0]), int(got["width"][0])) == (600, 1)
    _same(got, oracle_mod.search(y, block=1024, nwidths=3, threshold=1.0, return_stats=True))
    rng = np.random.default_rng(6)
    for nout in (1, 5, 31, 33, 255, 257):                  # rows shorter than a block / than the widest boxcar
        y = rng.normal(0, 1, size=(2, 260)).astype(np.float32)
        want = oracle_mod.search(y, nout=nout, block=256, nwidths=6, threshold=-1e30, return_stats=True)
        _same(_gpu_search(torch.from_numpy(y).cuda(), nout, 256, 6, -1e30), want)
    with pytest.raises(gsp.GspError):
        gsp.Search(4, 1000, 1000, 1000, 6, 5.0, 10)        # block must be a supported power of two
    with pytest.raises(gsp.GspError):
        gsp.Search(4, 1000, 1000, 1024, 7, 5.0, 10)        # widths up to 32


def test_search_on_dedispersed_crafts_slice_finds_the_injected_pulses(oracle_mod):
    """The path end to end on the device: gsp_dedisperse then gsp_search on d_out (no copy in between);
    the candidate list equals the oracle's search of the oracle's dedispersion, and the brightest
    injected pulse (E4) is among the candidates at its DM and arrival sample."""
    cfg = workloads.get_config("crafts")
    nsamp = (1 << 18) + 50000
    a = workloads.plan_args(cfg, nsamp=nsamp)
    a["dm_list"] = a["dm_list"][::8]                       # 128 DMs 0, 8, ... (keeps the oracle pass short)
    cfg["pulses"] = dict(kind="fixed", items=[dict(dm=512.0, width=8, amp=3.0, t0=100000),
                                              dict(dm=520.0, width=2, amp=6.0, t0=30000)])
    x = workloads.make_filterbank(cfg, device="cuda", nsamp=nsamp)
    s1, s2 = oracle_mod.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"], a["subband_dm"],
                                     a["dm_list"], 1)
    with gsp.Plan(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], nsamp, a["nsub"], a["subband_dm"], a["dm_list"],
                  1, "u8") as plan:
        y = torch.empty((plan.ndm, plan.out_pitch), dtype=torch.float32, device="cuda")
        plan.dedisperse(x, y, torch.cuda.current_stream().cuda_stream)
        got = _gpu_search(y, plan.nout, 1024, 6, 6.0, want_stats=False)
        y_or = oracle_mod.dedisperse(x.cpu().numpy(), s1, s2, 1, nthreads=oracle_mod.max_threads())
    want = oracle_mod.search(y_or, block=1024, nwidths=6, threshold=6.0)
    _same(got, want, stats=False)
    assert want["count"] >= 2
    hits = [(int(d), int(u), int(w)) for d, u, w in zip(got["dm"], got["sample"], got["width"])]
    assert any(d == 64 and abs(u - 100000) <= 2 and w == 8 for d, u, w in hits)     # DM 512 = row 64
    assert any(d == 65 and abs(u - 30000) <= 24 for d, u, w in hits)                # DM 520 = row 65
