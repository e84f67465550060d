// gsp_tables.cpp — host side of a plan: argument checks, the delay-table builder
// (include/gsp.h header comment; BASELINE.json north_star; rule R3 of DESIGN.md §3),
// output extents, and the tile geometry of the shared-memory stage-2 kernel.
// Pure host arithmetic: no CUDA runtime call in this file.

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <numeric>

#include "gsp_internal.h"

namespace gsp {

namespace {

// Dispersion constant of BASELINE.json north_star: seconds * MHz^2 / (pc cm^-3).
constexpr double kKdm = 4.148808e3;

inline double channel_centre_mhz(const gsp_plan &p, int c) { return p.f_top + p.chan_bw * (double)c; }

// Rule R3: evaluate in binary64 in the order written — square by multiplication,
// reciprocal by division, subtract, multiply by K*DM, divide by the sample time —
// then round half up with floor(x + 0.5).
inline int32_t shift_in_samples(double dm, double f_mhz, double f_ref_mhz, double sample_s) {
    const double recip_f = 1.0 / (f_mhz * f_mhz);
    const double recip_ref = 1.0 / (f_ref_mhz * f_ref_mhz);
    const double samples = (kKdm * dm) * (recip_f - recip_ref) / sample_s;
    return (int32_t)std::floor(samples + 0.5);
}

inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

// Alignment (in 32-bit words) of the bulk-copy windows: 16 bytes.
constexpr int kWindowAlignWords = 4;

}  // namespace

gsp_status validate_args(int nchan, double f_top, double chan_bw, double dt, int64_t nsamp,
                         int nsub, double subband_dm, const double *dm_list, int ndm,
                         int downsamp, int in_dtype) {
    if (!dm_list) return GSP_ERR_INVALID_ARG;
    if (nchan < 1 || nsub < 1 || nchan % nsub != 0) return GSP_ERR_INVALID_ARG;
    if (!(chan_bw < 0.0) || !std::isfinite(chan_bw) || !std::isfinite(f_top)) return GSP_ERR_INVALID_ARG;
    if (!(f_top + chan_bw * (double)(nchan - 1) > 0.0)) return GSP_ERR_INVALID_ARG;
    if (!(dt > 0.0) || !std::isfinite(dt)) return GSP_ERR_INVALID_ARG;
    if (ndm < 1 || downsamp < 1 || nsamp < 1) return GSP_ERR_INVALID_ARG;
    if (!(subband_dm >= 0.0) || !std::isfinite(subband_dm)) return GSP_ERR_INVALID_ARG;
    for (int d = 0; d < ndm; ++d)
        if (!(dm_list[d] >= 0.0) || !std::isfinite(dm_list[d])) return GSP_ERR_INVALID_ARG;
    if (in_dtype != GSP_U8 && in_dtype != GSP_F32) return GSP_ERR_INVALID_ARG;
    return GSP_OK;
}

void build_delay_tables(gsp_plan &p) {
    p.cps = p.nchan / p.nsub;
    p.s1.resize(p.nchan);
    p.s2.resize((size_t)p.ndm * p.nsub);
    const double f_band_top = channel_centre_mhz(p, 0);
    // stage 1: every channel against the top channel of its own subband, at subband_dm
    for (int s = 0; s < p.nsub; ++s) {
        const double f_sub_top = channel_centre_mhz(p, s * p.cps);
        for (int j = 0; j < p.cps; ++j) {
            const int c = s * p.cps + j;
            p.s1[c] = shift_in_samples(p.subband_dm, channel_centre_mhz(p, c), f_sub_top, p.dt);
        }
    }
    // stage 2: every subband top against the band top, per trial DM, in downsampled samples
    const double dt_ds = p.dt * (double)p.ds;
    for (int d = 0; d < p.ndm; ++d)
        for (int s = 0; s < p.nsub; ++s)
            p.s2[(size_t)d * p.nsub + s] =
                shift_in_samples(p.dm_list[d], channel_centre_mhz(p, s * p.cps), f_band_top, dt_ds);
    // trial DMs in ascending order (ties keep list order): neighbours share windows
    p.order.resize(p.ndm);
    std::iota(p.order.begin(), p.order.end(), 0);
    std::stable_sort(p.order.begin(), p.order.end(),
                     [&](int a, int b) { return p.dm_list[a] < p.dm_list[b]; });
}

gsp_status compute_extents(gsp_plan &p) {
    p.H1 = *std::max_element(p.s1.begin(), p.s1.end());
    p.H2 = *std::max_element(p.s2.begin(), p.s2.end());
    p.n1 = p.nsamp - (int64_t)p.H1;
    p.n1d = p.n1 > 0 ? p.n1 / p.ds : 0;
    p.nout = p.n1d - (int64_t)p.H2;
    p.halo = (int64_t)p.H1 + (int64_t)p.ds * (int64_t)p.H2;
    if (p.n1 <= 0 || p.nout <= 0) return GSP_ERR_TOO_SHORT;
    p.out_pitch = (p.nout + 31) / 32 * 32;  // rows start on 128-byte boundaries
    return GSP_OK;
}

// Window of subband s needed by DM block blk (sorted positions [blk*Q, blk*Q+Q)):
// words [wstart, wstart + wlen) relative to the tile origin u0, both multiples of 4
// so that the bulk copies are 16-byte aligned.
static void block_window(const gsp_plan &p, int Q, int M, int blk, int s, int &wstart, int &wlen) {
    int lo = INT32_MAX, hi = 0;
    for (int q = 0; q < Q; ++q) {
        const int dq = std::min(blk * Q + q, p.ndm - 1);
        const int v = p.s2[(size_t)p.order[dq] * p.nsub + s];
        lo = std::min(lo, v);
        hi = std::max(hi, v);
    }
    const int al = kWindowAlignWords;
    wstart = lo & ~(al - 1);
    wlen = round_up(M + hi - wstart, al);
}

void plan_stage2_tiling(gsp_plan &p, size_t smem_budget_bytes) {
    Stage2Tiling best;
    p.t2 = best;
    if (p.nsub % 4 != 0) return;
    const bool f32 = (p.dtype == GSP_F32);
    // uint8: the un-divided subband sums S' <= cps*255*ds are packed two per word while `flush` of them
    // still fit a 16-bit lane (flush = 4, 2 or 1 subbands between folds into the 32-bit accumulators);
    // larger sums (DownSamp 8 and up at 64 channels per subband, Tables 2-3 of the paper) are int32 operands
    int mode = S2_F32;
    if (!f32) {
        const int64_t smax = (int64_t)p.cps * 255 * p.ds;
        if ((int64_t)p.nchan * 255 * p.ds > INT32_MAX) return;
        mode = 4 * smax <= 65535 ? S2_PK4 : 2 * smax <= 65535 ? S2_PK2 : smax <= 65535 ? S2_PK1 : S2_I32;
    }
    const bool packed = mode <= S2_PK1;
    const int tpw = packed ? 2 : 1;

    // (DMs per warp, words per lane) instantiated in gsp_kernels.cu; 16 consumer warps.  `eff` = measured cost of an
    // operand read of the shape relative to the best one (config 2 / config 4 with every shape forced,
    // profiles/r2_summary.md): one DM per warp keeps more loads in flight per accumulator register, 8-word rows
    // pay the per-tile overheads four times as often.
    struct Cand {
        int dpw, wpl;
        double eff;
    };
    static const Cand cand_u8[] = {{1, 32, 1.000}, {1, 16, 1.000}, {2, 16, 1.032}, {2, 8, 1.056}, {4, 8, 1.138}, {1, 8, 1.54}};
    static const Cand cand_w32[] = {{1, 32, 1.00}, {2, 32, 1.03}, {1, 16, 1.03}, {2, 16, 1.04}, {4, 16, 1.09},
                                    {2, 8, 1.11},  {4, 8, 1.15},  {1, 8, 1.50}};
    const int ncand = packed ? 6 : 8;
    double best_cost = 1e300;
    for (int ci = 0; ci < ncand; ++ci) {
        const Cand &c = packed ? cand_u8[ci] : cand_w32[ci];
        Stage2Tiling t;
        t.Q = 16 * c.dpw;
        t.M = 32 * c.wpl;
        t.tpw = tpw;
        t.mode = mode;
        t.chunk = 4;
        t.nchunk = p.nsub / t.chunk;
        t.ndmblk = (p.ndm + t.Q - 1) / t.Q;
        t.ntile_t = (p.nout + tpw * (int64_t)t.M - 1) / (tpw * (int64_t)t.M);
        int64_t stage_words = 0;
        double fill = 0;
        for (int blk = 0; blk < t.ndmblk; ++blk)
            for (int ch = 0; ch < t.nchunk; ++ch) {
                int64_t words = 0;
                for (int k = 0; k < t.chunk; ++k) {
                    int ws, wl;
                    block_window(p, t.Q, t.M, blk, ch * t.chunk + k, ws, wl);
                    words += wl;
                }
                stage_words = std::max(stage_words, words);
                fill += (double)words;
            }
        t.stage_words = (int)stage_words;
        const size_t fixed = 256;  // mbarriers
        const size_t per_stage = (size_t)stage_words * 4;
        // pipeline depth: about 112 KB of windows in flight, 3 to 6 stages (measured: config 2's 28 KB stages run
        // 0.6 % faster four deep than six deep, the smaller stages of the fine-stepped and float32 plans 1.5-3 %
        // slower), never more than fits
        const size_t want_stages = std::min<size_t>(6, std::max<size_t>(3, (112 * 1024 + per_stage - 1) / std::max<size_t>(per_stage, 1)));
        int nstage = (int)std::min<size_t>(want_stages, (smem_budget_bytes - fixed) / std::max<size_t>(per_stage, 1));
        if (nstage < 2) continue;
        t.nstage = nstage;
        t.smem_bytes = fixed + per_stage * nstage;
        // cost per useful operand word: the reads of the padded tiles (padded DMs and the ragged last time tile
        // are wasted reads) at the shape's measured efficiency, the window fills at a fifth of a read (measured:
        // the bulk-copy writes mostly fall into the ~5 % of pipe slots LDS.32 cannot use), and the idle SMs of
        // the last wave of the persistent grid.
        const double useful = (double)p.ndm * p.nsub * (double)p.nout / (double)tpw;
        const double reads = (double)t.ndmblk * t.Q * p.nsub * (double)t.M * (double)t.ntile_t;
        const double fills = fill * (double)t.ntile_t;
        double cost = (reads * c.eff + 0.2 * fills) / useful;
        const double ntiles = (double)t.ntile_t * t.ndmblk, nsm = (double)std::max(p.sm_count, 1);
        cost *= std::ceil(ntiles / nsm) * nsm / ntiles;
        if (nstage < 3) cost *= 1.10;  // shallow pipelines expose copy latency
        if (cost < best_cost) {
            best_cost = cost;
            best = t;
            best.supported = true;
        }
    }
    p.t2 = best;
}

void build_stage2_tables(const gsp_plan &p, std::vector<int4> &prod, std::vector<int32_t> &offs,
                         std::vector<int32_t> &rows) {
    const Stage2Tiling &t = p.t2;
    prod.assign((size_t)t.ndmblk * p.nsub, make_int4(0, 0, 0, 0));
    offs.assign((size_t)t.ndmblk * t.Q * p.nsub, 0);
    rows.assign((size_t)t.ndmblk * t.Q, -1);
    for (int blk = 0; blk < t.ndmblk; ++blk) {
        for (int ch = 0; ch < t.nchunk; ++ch) {
            int boff = 0;
            for (int k = 0; k < t.chunk; ++k) {
                const int s = ch * t.chunk + k;
                int ws, wl;
                block_window(p, t.Q, t.M, blk, s, ws, wl);
                prod[(size_t)blk * p.nsub + s] = make_int4(ws, wl, boff, 0);
                for (int q = 0; q < t.Q; ++q) {
                    const int dq = blk * t.Q + q;
                    const int src = std::min(dq, p.ndm - 1);
                    const int v = p.s2[(size_t)p.order[src] * p.nsub + s];
                    offs[(size_t)dq * p.nsub + s] = boff + (v - ws);
                }
                boff += wl;
            }
        }
        for (int q = 0; q < t.Q; ++q) {
            const int dq = blk * t.Q + q;
            if (dq < p.ndm) rows[dq] = p.order[dq];
        }
    }
}

}  // namespace gsp
