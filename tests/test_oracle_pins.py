"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test names the pin of DESIGN.md §"Oracle pins" (P1-P12) it implements and
the mistake it is there to catch.  None of them re-types the oracle's own loops:
they use closed forms, textbook special cases, invariants, brute force with an
independently written one-stage sum, and the survey's independently computed tables.
"""
import os

import numpy as np
import pytest

import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _tables(oracle, cfg, plan=0, **over):
    a = workloads.plan_args(cfg, plan)
    a.update(over)
    return oracle.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"],
                               a["subband_dm"], a["dm_list"], a["downsamp"])


def _rand_tables(rng, nchan, nsub, ndm, max1, max2):
    s1 = rng.integers(0, max1 + 1, size=nchan).astype(np.int32)
    s2 = rng.integers(0, max2 + 1, size=(ndm, nsub)).astype(np.int32)
    return s1, s2


def _brute_one_stage(x, s1, s2, ds):
    """Independent statement: one-stage sum with composite shift s1[c] + ds*s2[d][sub(c)]
    (Algorithm 2, with delays := composite), then the mean over ds."""
    nsamp, nchan = x.shape
    ndm, nsub = s2.shape
    cps = nchan // nsub
    n1d = (nsamp - int(s1.max())) // ds
    nout = n1d - int(s2.max())
    y = np.zeros((ndm, nout), dtype=np.float64)
    xx = x.astype(np.float64)
    for d in range(ndm):
        for c in range(nchan):
            comp = int(s1[c]) + ds * int(s2[d, c // cps])
            for k in range(ds):
                y[d] += xx[comp + k: comp + k + ds * nout: ds, c]
    return (y / ds).astype(np.float32)


# ----------------------------------------------------------------------------- P1
@pytest.mark.parametrize("ds", [1, 2, 4])
@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
def test_p1_dm0_is_plain_channel_sum(oracle_mod, ds, dtype):
    """subband_dm = 0 and DM = 0 -> y[u] = mean_k sum_c x[u*ds+k][c]  (BJ check, A14)."""
    rng = np.random.default_rng(11)
    nsamp, nchan, nsub = 203, 32, 4
    x = rng.integers(0, 256, size=(nsamp, nchan)).astype(dtype)
    s1, s2 = oracle_mod.delay_tables(nchan, 1500.0, -10.0, 1e-4, nsub, 0.0, [0.0], ds)
    assert not s1.any() and not s2.any()
    y = oracle_mod.dedisperse(x, s1, s2, ds)
    n = nsamp // ds
    want = x[: n * ds].astype(np.float64).sum(axis=1).reshape(n, ds).mean(axis=1)
    assert y.shape == (1, n)
    np.testing.assert_array_equal(y[0], want.astype(np.float32))


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("ds", [1, 2, 3])
@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
def test_p2_two_stage_equals_one_stage_with_composite_shifts(oracle_mod, ds, dtype):
    """Catches a wrong subband index, transposed s2, dropped channel, bad ds stride."""
    rng = np.random.default_rng(100 + ds)
    nsamp, nchan, nsub, ndm = 400, 24, 6, 7
    s1, s2 = _rand_tables(rng, nchan, nsub, ndm, 17, 23)
    x = rng.integers(0, 256, size=(nsamp, nchan)).astype(dtype)
    y = oracle_mod.dedisperse(x, s1, s2, ds)
    want = _brute_one_stage(x, s1, s2, ds)
    np.testing.assert_array_equal(y, want)


def test_p2_on_real_tables_tiny(oracle_mod):
    cfg = workloads.get_config("tiny")
    s1, s2 = _tables(oracle_mod, cfg)
    x = workloads.make_filterbank(cfg).numpy()
    y = oracle_mod.dedisperse(x, s1, s2, 1)
    for d in (0, 7, 20, 31):
        want = _brute_one_stage(x, s1, s2[d:d + 1], 1)
        # nout of the single-row brute force is longer (its own H2); compare the common part
        np.testing.assert_array_equal(y[d], want[0, : y.shape[1]])


# ----------------------------------------------------------------------------- P3
def test_p3_composite_shift_within_one_sample_of_one_stage_at_subband_dm(oracle_mod):
    """At DM_d = DM_sub: |s1[c] + ds*s2[d][sub(c)] - rnd(one-stage delay)| <= 1  (A15-ii).
    The one-stage delay is evaluated here with numpy longdouble from the formula of
    BASELINE.json north_star — a sign error, swapped reference or wrong constant in the
    oracle breaks the bound by tens of samples."""
    nchan, nsub, f_top, bw, dt = 256, 16, 1500.0, -1.953125, 49.152e-6
    dm = 300.0
    for ds in (1, 2):
        s1, s2 = oracle_mod.delay_tables(nchan, f_top, bw, dt, nsub, dm, [dm], ds)
        f = np.longdouble(f_top) + np.arange(nchan, dtype=np.longdouble) * np.longdouble(bw)
        one = np.longdouble(4.148808e3) * dm * (f ** -2 - np.longdouble(f_top) ** -2) / dt
        comp = s1.astype(np.int64) + ds * s2[0][np.arange(nchan) // (nchan // nsub)]
        err = np.abs(comp - np.asarray(one, dtype=np.float64))
        # rounding in units of dt (stage 1) plus units of ds*dt (stage 2)
        assert err.max() <= 0.5 + 0.5 * ds + 1e-6
        assert one[-1] > 1000  # the sweep is really there


# ----------------------------------------------------------------------------- P4
def test_p4_linearity_exact(oracle_mod):
    rng = np.random.default_rng(4)
    cfg = workloads.get_config("tiny")
    s1, s2 = _tables(oracle_mod, cfg)
    nsamp = 4000
    x1 = rng.integers(0, 40, size=(nsamp, 64)).astype(np.uint8)
    x2 = rng.integers(0, 30, size=(nsamp, 64)).astype(np.uint8)
    y1 = oracle_mod.dedisperse(x1, s1, s2, 1)
    y2 = oracle_mod.dedisperse(x2, s1, s2, 1)
    y12 = oracle_mod.dedisperse((3 * x1 + 4 * x2).astype(np.uint8), s1, s2, 1)
    np.testing.assert_array_equal(y12, 3 * y1 + 4 * y2)


# ----------------------------------------------------------------------------- P5
@pytest.mark.parametrize("ds", [1, 2])
def test_p5_time_shift_equivariance(oracle_mod, ds):
    rng = np.random.default_rng(5)
    nchan, nsub, ndm = 16, 4, 5
    s1, s2 = _rand_tables(rng, nchan, nsub, ndm, 9, 12)
    x = rng.integers(0, 256, size=(300, nchan)).astype(np.uint8)
    m = 7
    xs = np.concatenate([np.zeros((m * ds, nchan), np.uint8), x])
    y = oracle_mod.dedisperse(x, s1, s2, ds)
    ys = oracle_mod.dedisperse(xs, s1, s2, ds)
    np.testing.assert_array_equal(ys[:, m: m + y.shape[1]], y)


# ----------------------------------------------------------------------------- P6
@pytest.mark.parametrize("ds", [1, 2, 4])
def test_p6_impulse_lands_where_the_tables_say(oracle_mod, ds):
    """x[t0][c0] = A -> row d has one non-zero A/ds at u = floor((t0 - s1[c0])/ds) - s2[d][sub(c0)]."""
    cfg = workloads.get_config("tiny")
    s1, s2 = _tables(oracle_mod, cfg, downsamp=ds)
    nsamp, t0, A = 8192, 5003, 200
    for c0 in (0, 13, 63):
        x = np.zeros((nsamp, 64), np.uint8)
        x[t0, c0] = A
        y = oracle_mod.dedisperse(x, s1, s2, ds)
        for d in range(s2.shape[0]):
            u = (t0 - int(s1[c0])) // ds - int(s2[d, c0 // 8])
            nz = np.flatnonzero(y[d])
            if 0 <= u < y.shape[1]:
                assert nz.tolist() == [u]
                assert y[d, u] == np.float32(A / ds)
            else:
                assert nz.size == 0


# ----------------------------------------------------------------------------- P7
@pytest.mark.parametrize("ds", [1, 2, 8])
def test_p7_constant_input(oracle_mod, ds):
    cfg = workloads.get_config("tiny")
    s1, s2 = _tables(oracle_mod, cfg, downsamp=ds)
    for v, dtype in ((255, np.uint8), (3, np.uint8), (1.5, np.float32)):
        x = np.full((8192, 64), v, dtype=dtype)
        y = oracle_mod.dedisperse(x, s1, s2, ds)
        assert np.all(y == np.float32(64 * v))


# ----------------------------------------------------------------------------- P8
@pytest.mark.parametrize("ds", [1, 2])
def test_p8_ramp_closed_form(oracle_mod, ds):
    """x[t][c] = t -> y_d[u] = sum_c (u*ds + (ds-1)/2 + s1[c] + ds*s2[d][sub(c)])."""
    cfg = workloads.get_config("tiny")
    s1, s2 = _tables(oracle_mod, cfg, downsamp=ds)
    nsamp = 8192
    x = np.repeat(np.arange(nsamp, dtype=np.float32)[:, None], 64, axis=1)
    y = oracle_mod.dedisperse(x, s1, s2, ds)
    u = np.arange(y.shape[1], dtype=np.float64)
    for d in (0, 5, 31):
        comp = s1.astype(np.float64) + ds * s2[d][np.arange(64) // 8]
        want = 64 * (u * ds + (ds - 1) / 2.0) + comp.sum()
        np.testing.assert_array_equal(y[d], want.astype(np.float32))


# ----------------------------------------------------------------------------- P9
@pytest.mark.parametrize("name", ["tiny", "crafts", "uwb"])
def test_p9_table_structure(oracle_mod, name):
    cfg = workloads.get_config(name)
    s1, s2 = _tables(oracle_mod, cfg)
    nsub = s2.shape[1]
    cps = cfg["nchan"] // nsub
    s1r = s1.reshape(nsub, cps)
    assert np.all(s1r[:, 0] == 0)
    assert np.all(np.diff(s1r, axis=1) >= 0)
    assert np.all(s2[:, 0] == 0)
    assert np.all(s2[0] == 0)                 # DM 0
    assert np.all(np.diff(s2, axis=0) >= 0)   # sorted DM list
    assert np.all(np.diff(s2, axis=1) >= 0)
    assert s1.min() >= 0 and s2.min() >= 0


# ----------------------------------------------------------------------------- P10
@pytest.mark.parametrize("ds", [1, 2])
def test_p10_block_carry_concatenation_equals_one_shot(oracle_mod, ds):
    """Algorithm 1's lastdata/data carry: blocks with the max-delay
    tail prepended reproduce the one-shot output."""
    rng = np.random.default_rng(10)
    nchan, nsub, ndm = 16, 4, 6
    s1, s2 = _rand_tables(rng, nchan, nsub, ndm, 11, 9)
    H1, H2 = int(s1.max()), int(s2.max())
    H = H1 + ds * H2
    B, nblk = 64, 5
    x = rng.integers(0, 256, size=(B * nblk, nchan)).astype(np.uint8)
    full = oracle_mod.dedisperse(x, s1, s2, ds)
    first = oracle_mod.dedisperse(x[:B], s1, s2, ds)
    nout0 = first.shape[1]
    parts = [first]
    for k in range(1, nblk):
        start = ds * nout0 + (k - 1) * B
        blk = x[start: start + B + H]
        yk = oracle_mod.dedisperse(blk, s1, s2, ds)
        assert yk.shape[1] == B // ds
        parts.append(yk)
    cat = np.concatenate(parts, axis=1)
    np.testing.assert_array_equal(cat, full[:, : cat.shape[1]])
    assert full.shape[1] - cat.shape[1] < max(ds, 1) + 1


# ----------------------------------------------------------------------------- P11
def _read_rows(fname):
    rows = []
    with open(os.path.join(GOLD, fname)) as fh:
        for line in fh:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


@pytest.mark.parametrize("row", _read_rows("tiny_pulse.txt"), ids=lambda r: r[0])
def test_p11_tiny_injected_pulse_peaks_at_true_dm_and_arrival(oracle_mod, row):
    """The generator injects with its own copy of the dispersion law; the oracle must
    put the peak at DM 100 (index 20) and at the arrival sample (A16)."""
    _, sub_dm, vmax, d_idx, u_first, u_last = row
    cfg = workloads.get_config("tiny")
    s1, s2 = _tables(oracle_mod, cfg, subband_dm=float(sub_dm))
    x = workloads.make_filterbank(cfg, noise=False).numpy()
    y = oracle_mod.dedisperse(x, s1, s2, 1)
    assert y.max() == float(vmax)
    d, u = np.unravel_index(np.argmax(y), y.shape)   # first argmax in C order
    assert d == int(d_idx)
    where = np.flatnonzero(y[d] == y.max())
    assert where.min() == int(u_first)
    if int(u_last) >= 0:
        assert where.max() == int(u_last)
    assert where.max() - where.min() < 4          # inside the 4-sample top-hat
    assert u == int(u_first)
    # and no other DM row reaches the maximum
    rows_at_max = np.flatnonzero((y == y.max()).any(axis=1))
    assert rows_at_max.tolist() == [int(d_idx)]


def test_p11_noisy_matched_plan_detects_pulse(oracle_mod):
    """With DM_sub = 100 the noisy Tiny input peaks at DM 100 near sample 3001 (z ~ 18)."""
    cfg = workloads.get_config("tiny")
    s1, s2 = _tables(oracle_mod, cfg, subband_dm=100.0)
    x = workloads.make_filterbank(cfg).numpy()
    y = oracle_mod.dedisperse(x, s1, s2, 1)
    z = (y - y.mean(axis=1, keepdims=True)) / y.std(axis=1, keepdims=True)
    d, u = np.unravel_index(np.argmax(z), z.shape)
    assert d == 20 and abs(int(u) - 3001) <= 2 and z[d, u] > 10


# ----------------------------------------------------------------------------- P12
@pytest.mark.parametrize("row", _read_rows("table_extents.txt"), ids=lambda r: f"{r[0]}{r[1]}")
def test_p12_table_extents_match_survey(oracle_mod, row):
    name, plan, H1, H2, nout, sum1, sum2 = row[0], *map(int, row[1:])
    cfg = workloads.get_config(name)
    s1, s2 = _tables(oracle_mod, cfg, plan)
    g = oracle_mod.geometry(cfg["nsamp"], s1, s2, cfg["plans"][plan]["downsamp"])
    assert (g["H1"], g["H2"], g["nout"]) == (H1, H2, nout)
    if sum1 >= 0:
        assert int(s1.sum()) == sum1 and int(s2.astype(np.int64).sum()) == sum2


def test_p12_tiny_rows_match_survey(oracle_mod):
    cfg = workloads.get_config("tiny")
    s1, s2 = _tables(oracle_mod, cfg)
    rows = {r[0]: list(map(int, r[1:])) for r in _read_rows("tiny_tables.txt")}
    assert s2[20].tolist() == rows["s2_dm100"]
    assert s2[31].tolist() == rows["s2_dm155"]
    assert s1[56:64].tolist() == rows["s1_56_63"]


# ----------------------------------------------------------------------------- P13 + misc
def test_p13_exactness_headroom():
    assert 4096 * 255 < 2 ** 24 and 64 * 255 < 2 ** 16 and 32 * 255 * 2 < 2 ** 16


def test_points_agree_with_full_matrix(oracle_mod):
    """The per-point routine (used at benchmark sizes) and the full routine are two
    statements of the same definition; they must agree bit for bit."""
    rng = np.random.default_rng(77)
    for ds, dtype in ((1, np.uint8), (2, np.uint8), (4, np.float32)):
        s1, s2 = _rand_tables(rng, 32, 8, 9, 13, 21)
        x = rng.normal(100, 20, size=(500, 32)).clip(0, 255).astype(dtype)
        y = oracle_mod.dedisperse(x, s1, s2, ds)
        d = rng.integers(0, 9, size=64)
        u = rng.integers(0, y.shape[1], size=64)
        p = oracle_mod.points(x, s1, s2, ds, d, u)
        np.testing.assert_array_equal(p, y[d, u])


@pytest.mark.parametrize("ds", [1, 2, 4])
@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
def test_points_pinned_directly_to_the_one_stage_brute_force(oracle_mod, ds, dtype):
    """oracle.points carries the full-size parity of configs 2-5: pin it DIRECTLY (not through
    oracle.dedisperse) to the independent numpy one-stage brute force with composite shifts
    (Algorithm 2; SURVEY §8(c) O4-O6 / pin P2), on the REAL Tiny tables
    (rule R3, 64 channels, 8 subbands, 32 DMs) built for downsamp 1, 2 and 4."""
    cfg = workloads.get_config("tiny")
    a = workloads.plan_args(cfg)
    s1, s2 = oracle_mod.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"], a["subband_dm"],
                                     a["dm_list"], ds)
    assert s1.max() == 323 and s2.max() == {1: 2887, 2: 1444, 4: 722}[ds]
    x = workloads.make_filterbank(cfg).numpy()
    if dtype == np.float32:
        x = (x.astype(np.float32) - 128.0) / 16.0 + np.float32(0.125)
    rng = np.random.default_rng(5 + ds)
    nout = (x.shape[0] - 323) // ds - int(s2.max())
    for d in (0, 1, 13, 20, 31):
        want = _brute_one_stage(x, s1, s2[d:d + 1], ds)[0]
        u = np.unique(np.concatenate([[0, nout - 1], rng.integers(0, nout, size=200)]))
        got = oracle_mod.points(x, s1, s2, ds, np.full(u.size, d), u)
        if dtype == np.uint8:
            np.testing.assert_array_equal(got, want[u])
        else:   # binary64 sums in two different orders, each rounded once to float32
            np.testing.assert_allclose(got, want[u], rtol=0, atol=2e-6 * float(np.abs(want).max()))


def test_f32_oracle_matches_u8_oracle_on_integer_data(oracle_mod):
    rng = np.random.default_rng(78)
    s1, s2 = _rand_tables(rng, 32, 4, 5, 10, 15)
    x = rng.integers(0, 256, size=(300, 32)).astype(np.uint8)
    for ds in (1, 2):
        np.testing.assert_array_equal(oracle_mod.dedisperse(x, s1, s2, ds),
                                      oracle_mod.dedisperse(x.astype(np.float32), s1, s2, ds))


def test_f32_accumulates_in_binary64(oracle_mod):
    """Large cancelling terms: a float32 accumulator would lose the small term."""
    x = np.zeros((4, 4), np.float32)
    x[:, 0], x[:, 1], x[:, 2], x[:, 3] = 1e8, 1.0, -1e8, 0.25
    s1 = np.zeros(4, np.int32)
    s2 = np.zeros((1, 1), np.int32)
    y = oracle_mod.dedisperse(x, s1, s2, 1)
    assert np.all(y == np.float32(1.25))


def test_threads_do_not_change_result(oracle_mod):
    rng = np.random.default_rng(79)
    s1, s2 = _rand_tables(rng, 32, 4, 12, 10, 15)
    x = rng.normal(0, 1, size=(600, 32)).astype(np.float32)
    a = oracle_mod.dedisperse(x, s1, s2, 2, nthreads=1)
    b = oracle_mod.dedisperse(x, s1, s2, 2, nthreads=4)
    np.testing.assert_array_equal(a, b)


def test_too_short_input_is_rejected(oracle_mod):
    cfg = workloads.get_config("tiny")
    s1, s2 = _tables(oracle_mod, cfg)
    with pytest.raises(ValueError):
        oracle_mod.dedisperse(np.zeros((3000, 64), np.uint8), s1, s2, 1)
