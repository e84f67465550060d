"""Pins of the oracle's RFI prologue (readings F1-F4) and single-pulse search (readings S1-S6):
the paper names both steps and prints no mechanics, so DESIGN.md §3a is the
specification; these tests tie the C++ oracle to things that are not itself — closed forms, numpy
restatements written in a different shape (Python big integers, cumulative sums in binary64),
invariants and degenerate cases — chosen so that a dropped term, a wrong sign, an off-by-one index
or a swapped tie-break fails one of them.  CPU only.
"""
import math

import numpy as np
import pytest


# ============================================================================== RFI prologue
def _numpy_rfi(x, mask, pad, sigma, B):
    """Independent restatement with Python integers and fractions-free integer algebra:
    clipped  <=>  d > 0 and d*d > sigma^2 * V  is NOT used (it would square sigma); instead the
    oracle's own binary64 comparison is reproduced from exact integers with math.sqrt (IEEE)."""
    x1 = x.copy()
    if mask is not None:
        x1[:, mask.astype(bool)] = pad[mask.astype(bool)][None, :]
    z = [int(v) for v in x1.astype(np.int64).sum(axis=1)]
    clipped = np.zeros(len(z), dtype=bool)
    if sigma > 0:
        for t0 in range(0, len(z), B):
            blk = z[t0:t0 + B]
            n, S1, S2 = len(blk), sum(blk), sum(v * v for v in blk)
            rhs = sigma * math.sqrt(float(n * S2 - S1 * S1))
            for i, v in enumerate(blk):
                clipped[t0 + i] = float(n * v - S1) > rhs
    x2 = x1.copy()
    x2[clipped] = pad[None, :]
    return x2, np.array(z, dtype=np.int64), clipped


def test_rfi_identity_without_mask_and_clip(oracle_mod):
    rng = np.random.default_rng(0)
    x = rng.integers(0, 256, size=(700, 48), dtype=np.uint8)
    x2, z, c = oracle_mod.rfi_prologue(x, None, np.zeros(48, np.uint8))
    np.testing.assert_array_equal(x2, x)
    np.testing.assert_array_equal(z, x.astype(np.int64).sum(axis=1))
    assert not c.any()


def test_rfi_channel_mask_replaces_exactly_the_masked_channels(oracle_mod):
    rng = np.random.default_rng(1)
    x = rng.integers(0, 256, size=(300, 64), dtype=np.uint8)
    mask = (rng.random(64) < 0.25).astype(np.uint8)
    pad = rng.integers(0, 256, size=64, dtype=np.uint8)
    x2, z, c = oracle_mod.rfi_prologue(x, mask, pad)
    want = np.where(mask[None, :].astype(bool), pad[None, :], x)
    np.testing.assert_array_equal(x2, want)
    np.testing.assert_array_equal(z, want.astype(np.int64).sum(axis=1))
    assert not c.any() and mask.sum() > 3


@pytest.mark.parametrize("sigma,expect", [(7.0, True), (7.9, True), (8.0, False), (30.0, False)])
def test_rfi_clip_closed_form_constant_plus_burst(oracle_mod, sigma, expect):
    """Constant input v with K burst rows raised by a, block of n rows:  n*z - S1 = nchan*a*(n-K) on the
    burst rows, n*S2 - S1^2 = (nchan*a)^2 * K*(n-K)  =>  clipped iff sqrt((n-K)/K) > sigma (7.94 here)."""
    n, K, nchan, v, a = 256, 4, 32, 100, 20
    x = np.full((3 * n, nchan), v, dtype=np.uint8)
    burst = np.array([n + 5, n + 6, n + 100, n + 255])          # all in the middle block
    x[burst] += a
    pad = np.full(nchan, 7, dtype=np.uint8)
    x2, z, c = oracle_mod.rfi_prologue(x, None, pad, clip_sigma=sigma, clip_block=n)
    assert math.sqrt((n - K) / K) > 7.9 and math.sqrt((n - K) / K) < 8.0
    want = np.zeros(3 * n, dtype=bool)
    if expect:
        want[burst] = True
    np.testing.assert_array_equal(c.astype(bool), want)
    np.testing.assert_array_equal(x2[want], np.broadcast_to(pad, (int(want.sum()), nchan)))
    np.testing.assert_array_equal(x2[~want], x[~want])


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_rfi_matches_the_integer_restatement_on_noise_with_bursts(oracle_mod, seed):
    rng = np.random.default_rng(seed)
    nsamp, nchan, B = 3000, 96, 512            # ragged last block (3000 = 5*512 + 440)
    x = rng.normal(128, 12, size=(nsamp, nchan)).round().clip(0, 255).astype(np.uint8)
    for t in rng.integers(0, nsamp, 12):
        x[t] = np.minimum(255, x[t].astype(int) + rng.integers(5, 60)).astype(np.uint8)
    mask = (rng.random(nchan) < 0.1).astype(np.uint8)
    pad = rng.integers(100, 160, size=nchan, dtype=np.uint8)
    got = oracle_mod.rfi_prologue(x, mask, pad, clip_sigma=3.0, clip_block=B)
    want = _numpy_rfi(x, mask, pad, 3.0, B)
    np.testing.assert_array_equal(got[1], want[1])
    np.testing.assert_array_equal(got[2].astype(bool), want[2])
    np.testing.assert_array_equal(got[0], want[0])
    assert 3 <= want[2].sum() <= 60          # the bursts (and little else) were clipped


def test_rfi_all_channels_masked_gives_constant_dedispersed_output(oracle_mod):
    """Everything replaced by pad -> constant filterbank -> y = sum(pad) for every DM and sample (pin P7)."""
    rng = np.random.default_rng(3)
    x = rng.integers(0, 256, size=(4000, 32), dtype=np.uint8)
    pad = rng.integers(0, 256, size=32, dtype=np.uint8)
    x2, _, _ = oracle_mod.rfi_prologue(x, np.ones(32, np.uint8), pad)
    s1, s2 = oracle_mod.delay_tables(32, 1500.0, -4.0, 1e-4, 4, 30.0, [0.0, 20.0, 60.0], 1)
    y = oracle_mod.dedisperse(x2, s1, s2, 1)
    assert np.all(y == np.float32(pad.astype(np.int64).sum()))


def test_rfi_rejects_blocks_that_overflow_the_exact_integers(oracle_mod):
    x = np.zeros((10, 4096), dtype=np.uint8)
    with pytest.raises(ValueError):
        oracle_mod.rfi_prologue(x, None, np.zeros(4096, np.uint8), clip_sigma=3.0, clip_block=4096)


# ============================================================================== single-pulse search
def _numpy_search(y, L, nwidths, thr):
    """Restatement in binary64 with cumulative sums (a different shape of the same definition): block
    mean / std by numpy, boxcars as differences of a cumulative sum.  Agrees with the float32 tree of the
    oracle to ~1e-5 relative, so it pins values within a tolerance and the argmax wherever the runner-up is
    further away than that."""
    ndm, nout = y.shape
    nblk = -(-nout // L)
    res = []
    for d in range(ndm):
        z = np.empty(nout)
        for b in range(nblk):
            seg = y[d, b * L:(b + 1) * L].astype(np.float64)
            sd = seg.std()
            z[b * L:(b + 1) * L] = (seg - seg.mean()) / sd if sd > 0 else 0.0
        cs = np.concatenate([[0.0], np.cumsum(z)])
        snr = np.full((nwidths, nout), -np.inf)
        for j in range(nwidths):
            w = 1 << j
            if w <= nout:
                snr[j, : nout - w + 1] = (cs[w:] - cs[:-w]) / math.sqrt(w)
        for b in range(nblk):
            blk = snr[:, b * L:(b + 1) * L]
            j, i = np.unravel_index(np.argmax(blk), blk.shape)
            srt = np.sort(blk.ravel())
            res.append((d, b, b * L + i, 1 << j, blk[j, i], srt[-1] - srt[-2]))
    return res


def test_search_constant_input_gives_no_candidate(oracle_mod):
    y = np.full((3, 5000), 524288.0, dtype=np.float32)
    r = oracle_mod.search(y, block=1024, threshold=1e-3)
    assert r["count"] == 0


def test_search_constant_block_semantics_as_gsp_h_states_them(oracle_mod):
    """include/gsp.h: a constant block has r_f = 0 and z = 0, so its winner is (snr 0, width 1, first sample)
    — a candidate iff threshold <= 0 — unless a boxcar that starts in it reaches a pulse in the next block."""
    L = 256
    y = np.full((1, 3 * L), 7.0, dtype=np.float32)
    r = oracle_mod.search(y, block=L, nwidths=6, threshold=0.0, return_stats=True)
    assert r["count"] == 3 and list(r["sample"]) == [0, L, 2 * L] and list(r["width"]) == [1, 1, 1]
    assert list(r["snr"]) == [0.0, 0.0, 0.0] and np.all(r["stats"][0, :, 1] == 0.0)
    assert oracle_mod.search(y, block=L, nwidths=6, threshold=1e-30)["count"] == 0
    # block 0 constant, a top-hat of A on the first two samples of block 1 (otherwise zero):
    #   mu1 = 2A/L, var1 = 2A^2/L - mu1^2, z[L] = z[L+1] = (A - mu1)/sigma1 =: zp, z elsewhere in block 1 < 0.
    #   boxcars starting in block 0: width 2 at L-1 sums z[L-1] + z[L] = zp      -> snr = zp * 0.70710678f
    #                                width 4 at L-2 sums 0 + 0 + zp + zp = 2 zp -> snr = 2 zp * 0.5 = zp  (best)
    #                                width 4 at L-3 -> zp * 0.5; width 8 at L-6 .. L-7 -> 2 zp * 0.35355339f
    A = 100.0
    y = np.full((1, 2 * L), 7.0, dtype=np.float32)
    y[0, L:] = 0.0
    y[0, L:L + 2] = A
    mu1 = 2 * A / L
    zp = np.float32(np.float32(A - np.float32(mu1)) * np.float32(1.0 / math.sqrt(2 * A * A / L - mu1 * mu1)))
    r = oracle_mod.search(y, block=L, nwidths=6, threshold=5.0)
    assert r["count"] == 2
    assert (int(r["sample"][0]), int(r["width"][0])) == (L - 2, 4)             # the constant block's winner
    assert r["snr"][0] == np.float32(np.float32(zp + zp) * np.float32(0.5))
    assert (int(r["sample"][1]), int(r["width"][1])) == (L, 2)                 # the pulse's own block
    assert r["snr"][1] == np.float32(np.float32(zp + zp) * np.float32(0.70710678))


def test_search_block_statistics_are_exact_on_integer_data(oracle_mod):
    """Integer-valued rows (the uint8 path): the tree sums are exact, so mu_f and r_f equal the float32
    roundings of the binary64 values computed from exact integer sums."""
    rng = np.random.default_rng(4)
    y = rng.integers(500000, 540000, size=(2, 3000)).astype(np.float32)
    st = oracle_mod.search(y, block=1024, threshold=100.0, return_stats=True)["stats"]
    for d in range(2):
        for b in range(3):
            seg = [int(v) for v in y[d, b * 1024:(b + 1) * 1024]]
            n, S1, S2 = len(seg), sum(seg), sum(v * v for v in seg)
            mu = float(S1) / n
            var = float(S2) / n - mu * mu
            assert st[d, b, 0] == np.float32(mu)
            assert st[d, b, 1] == np.float32(1.0 / math.sqrt(var))
    assert len(seg) == 3000 - 2048         # the ragged block divides by its own length


def test_search_tree_sum_order_is_the_stated_one(oracle_mod):
    """S1's summation ORDER (P:86 gives no mechanics): a perfect binary tree over the block's
    slots in natural order.  The vectors are float32-exact and chosen so that the three plausible orders
    round to DIFFERENT float32 means, worked out by hand here (2^53 + 1 ties to even = 2^53 in binary64):
      row A = [1, 2^53, 1, -2^53], block 4
        natural tree   (1 + 2^53) + (1 - 2^53) = 2^53 - (2^53 - 1) = 1      -> mu = 0.25
        left to right  ((1 + 2^53) + 1) - 2^53 = 2^53 - 2^53       = 0      -> mu = 0
      row B = [2^53, 1, -2^53, 1, 0, 0, 0, 0], block 8
        natural tree   ((2^53 + 1) + (-2^53 + 1)) + 0 = 2^53 - (2^53 - 1) = 1       -> mu = 0.125
        strided tree   ((a0+a4) + (a2+a6)) + ((a1+a5) + (a3+a7)) = 0 + 2  = 2       -> mu = 0.25
    A sequential-sum oracle fails row A, a stride-first butterfly fails row B."""
    P = 2.0 ** 53
    row_a = np.array([1.0, P, 1.0, -P], dtype=np.float32)
    assert [float(v) for v in row_a] == [1.0, P, 1.0, -P]                    # exact in float32
    st = oracle_mod.search(row_a[None, :].copy(), block=4, nwidths=1, threshold=1e30, return_stats=True)["stats"]
    assert st[0, 0, 0] == np.float32(0.25)
    row_b = np.array([P, 1.0, -P, 1.0, 0.0, 0.0, 0.0, 0.0], dtype=np.float32)
    st = oracle_mod.search(row_b[None, :].copy(), block=8, nwidths=1, threshold=1e30, return_stats=True)["stats"]
    assert st[0, 0, 0] == np.float32(0.125)
    # S2's formula on a row whose sums can be followed by hand: v = [1, 2^27, 1, 2^27], squares 1, 2^54, 1, 2^54;
    #   S1 = 2^28 + 2 (exact), mu = 2^26 + 0.5;  S2 = (1 + 2^54) + (1 + 2^54) = 2^55 (each one is lost);
    #   var = S2/4 - fl(mu*mu), multiply and subtract rounded separately (no FMA)
    row_c = np.array([1.0, 2.0 ** 27, 1.0, 2.0 ** 27], dtype=np.float32)
    st = oracle_mod.search(row_c[None, :].copy(), block=4, nwidths=1, threshold=1e30, return_stats=True)["stats"]
    mu = (2.0 + 2.0 ** 28) / 4
    var = 2.0 ** 55 / 4 - mu * mu
    assert st[0, 0, 0] == np.float32(mu) and st[0, 0, 1] == np.float32(1.0 / math.sqrt(var))


def test_search_tree_sum_is_a_harmless_ordering_of_the_plain_statistic(oracle_mod):
    """The tree is a reading of a step the paper leaves open; it must not be a different
    statistic.  On non-integer float32 rows (the float32 path, where the order matters) mu_f and r_f must
    agree with the EXACTLY rounded sums (math.fsum; the squares of float32 values are exact in binary64)
    to within one float32 ulp, ragged last block included."""
    rng = np.random.default_rng(11)
    L, nout = 1024, 3 * 1024 + 333
    y = (rng.normal(1000.0, 37.0, size=(3, nout)) * rng.uniform(0.5, 2.0, size=(3, 1))).astype(np.float32)
    st = oracle_mod.search(y, block=L, nwidths=1, threshold=1e30, return_stats=True)["stats"]
    worst = 0.0
    for d in range(3):
        for b in range(4):
            seg = [float(v) for v in y[d, b * L:(b + 1) * L]]
            n = len(seg)
            mu = math.fsum(seg) / n
            var = math.fsum(v * v for v in seg) / n - mu * mu
            r = 1.0 / math.sqrt(var)
            for got, want in ((st[d, b, 0], mu), (st[d, b, 1], r)):
                ulp = float(np.spacing(np.float32(abs(want))))
                worst = max(worst, abs(float(got) - want) / ulp)
    assert n == 333
    assert worst <= 1.0, worst


def test_search_recovers_an_injected_pulse_closed_form(oracle_mod):
    """One top-hat of width w and height A on a zero row: mu = A*w/L, var = A^2*w/L - mu^2, and the best
    boxcar is the width-w one starting at the pulse: snr = w*(A - mu)/sigma/sqrt(w)."""
    L, w, A, u0 = 1024, 8, 50.0, 1024 + 300
    y = np.zeros((5, 4096), dtype=np.float32)
    y[2, u0:u0 + w] = A
    r = oracle_mod.search(y, block=L, nwidths=6, threshold=5.0)
    assert r["count"] == 1
    assert (int(r["dm"][0]), int(r["sample"][0]), int(r["width"][0])) == (2, u0, w)
    mu = A * w / L
    sigma = math.sqrt(A * A * w / L - mu * mu)
    want = w * (A - mu) / sigma / math.sqrt(w)
    assert abs(float(r["snr"][0]) - want) <= 2e-5 * want


@pytest.mark.parametrize("w", [1, 2, 4, 16, 32])
def test_search_picks_the_matching_width(oracle_mod, w):
    rng = np.random.default_rng(w)
    y = rng.normal(0, 1, size=(1, 2048)).astype(np.float32)
    y[0, 700:700 + w] += 12.0 / math.sqrt(w) + 3.0
    r = oracle_mod.search(y, block=1024, nwidths=6, threshold=8.0)
    assert r["count"] == 1 and int(r["width"][0]) == w and abs(int(r["sample"][0]) - 700) <= max(1, w // 4)


def test_search_matches_cumsum_restatement_on_noise(oracle_mod):
    rng = np.random.default_rng(9)
    ndm, nout, L, nw = 4, 5000, 512, 6
    y = (rng.normal(0, 30, size=(ndm, nout)) + 5000).astype(np.float32)
    for d in range(ndm):
        y[d, 400 + 900 * d: 400 + 900 * d + (1 << d)] += 150.0
    got = oracle_mod.search(y, block=L, nwidths=nw, threshold=-1e9)          # every block reports its best
    want = _numpy_search(y, L, nw, -1e9)
    assert got["count"] == len(want) == ndm * 10
    for k, (d, b, u, w, snr, margin) in enumerate(want):
        assert int(got["dm"][k]) == d
        assert abs(float(got["snr"][k]) - snr) <= 3e-5 * max(1.0, abs(snr))
        if margin > 1e-3:
            assert (int(got["sample"][k]), int(got["width"][k])) == (u, w)
        assert b * L <= int(got["sample"][k]) < (b + 1) * L


def test_search_boxcar_crosses_block_boundaries_but_not_the_end(oracle_mod):
    """A width-32 pulse straddling a block boundary is found from its START block; no boxcar reads past nout."""
    nout = 2048 + 200
    y = np.zeros((1, nout), dtype=np.float32)
    y[0, 1024 - 16: 1024 + 16] = 10.0
    y[0, nout - 7: nout] = 10.0                   # 7 samples at the very end of the ragged last block
    r = oracle_mod.search(y, block=1024, nwidths=6, threshold=3.0)
    starts = {int(b) for b in r["sample"]}
    assert 1024 - 16 in starts                    # the straddling pulse, reported by block 0
    last = [k for k in range(len(r["sample"])) if r["sample"][k] >= 2048]
    assert len(last) == 1 and nout - 8 <= int(r["sample"][last[0]])
    assert int(r["sample"][last[0]]) + int(r["width"][last[0]]) <= nout


def test_search_tie_breaks_smaller_width_then_earlier_sample(oracle_mod):
    y = np.zeros((1, 1024), dtype=np.float32)
    y[0, 100] = 8.0
    y[0, 500] = 8.0                               # identical pulses: the earlier one wins
    r = oracle_mod.search(y, block=1024, nwidths=3, threshold=1.0)
    assert (int(r["sample"][0]), int(r["width"][0])) == (100, 1)
    # an exact tie between two widths: four samples of 1025 and one of 2044 on zeros give mu = 6 exactly,
    # z_p = fl(1019 r), z_q = fl(2038 r) = 2 z_p, so snr_2(pulse p) = 4 z_p * 0.5 == z_q = snr_0(sample q);
    # the smaller width wins although it comes later in time
    y = np.zeros((1, 1024), dtype=np.float32)
    y[0, 200:204] = 1025.0
    y[0, 600] = 2044.0
    r = oracle_mod.search(y, block=1024, nwidths=3, threshold=1.0, return_stats=True)
    assert r["stats"][0, 0, 0] == 6.0
    assert (int(r["sample"][0]), int(r["width"][0])) == (600, 1)
    assert float(r["snr"][0]) == float(np.float32(1019.0) * r["stats"][0, 0, 1]) * 2.0
    y[0, 600] = 2043.0                            # just below the tie: the width-4 boxcar wins
    r = oracle_mod.search(y, block=1024, nwidths=3, threshold=1.0)
    assert (int(r["sample"][0]), int(r["width"][0])) == (200, 4)


def test_search_threshold_is_monotone_and_order_is_dm_then_block(oracle_mod):
    rng = np.random.default_rng(11)
    y = rng.normal(0, 1, size=(6, 8192)).astype(np.float32)
    lo = oracle_mod.search(y, block=256, threshold=3.0)
    hi = oracle_mod.search(y, block=256, threshold=4.0)
    assert 0 < hi["count"] < lo["count"]
    key = lambda r: list(zip(r["dm"].tolist(), (r["sample"] // 256).tolist()))
    assert key(lo) == sorted(key(lo)) and set(key(hi)) <= set(key(lo))
    cap = oracle_mod.search(y, block=256, threshold=3.0, max_cand=5)
    assert cap["count"] == lo["count"] and len(cap["dm"]) == 5
    np.testing.assert_array_equal(cap["sample"], lo["sample"][:5])


def test_search_is_block_shift_equivariant(oracle_mod):
    """Prepending one whole block of samples moves every candidate by exactly L (same statistics per block)."""
    rng = np.random.default_rng(12)
    L = 512
    y = rng.normal(0, 1, size=(2, 4 * L)).astype(np.float32)
    y2 = np.concatenate([rng.normal(0, 1, size=(2, L)).astype(np.float32), y], axis=1)
    a = oracle_mod.search(y, block=L, threshold=-1e9)
    b = oracle_mod.search(y2, block=L, threshold=-1e9)
    keep = b["sample"] >= L
    # the last block of the shorter series ends at nout in both cases; block 0 of y2 may reach into y: drop it
    np.testing.assert_array_equal(b["sample"][keep] - L, a["sample"])
    np.testing.assert_array_equal(b["snr"][keep], a["snr"])
