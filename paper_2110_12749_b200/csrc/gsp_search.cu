// gsp_search.cu — single-pulse search on the dedispersed series, on the GPU.
//
// The step that follows dedispersion in the GSP pipeline ("pulsar search (RFI mitigation,
// de-dispersion and single-pulse search)"; run on the CPU in the paper).
// The paper prints no mechanics; this file computes readings S1-S6 of DESIGN.md §3a:
//
//   S1  blocks of L = 2^k samples per DM row; S1 = sum y, S2 = sum y^2 in binary64, added in a perfect
//       binary tree over the block's slots in natural order (absent slots of the ragged last block = 0)
//   S2  mu = S1/n, var = S2/n - mu*mu (no FMA), r = var > 0 ? 1/sqrt(var) : 0, mu_f = (float)mu, r_f = (float)r
//   S3  z[u] = (y[u] - mu_f) * r_f in float32, each sample with its own block's statistics
//   S4  boxcars of widths 2^j: B_0 = z, B_{j+1}[u] = B_j[u] + B_j[u + 2^j] (float32), valid while the window
//       ends at or before nout; snr_j[u] = B_j[u] * 2^(-j/2) (float32 constants)
//   S5  per (DM, block): the best (snr, j, u), larger snr first, then smaller j, then smaller u
//   S6  candidate iff snr >= threshold; candidates are listed in (DM, block) order
//
// Kernel layout.  One thread owns 8 consecutive samples; a CTA of L/8 threads owns one DM row and a run
// of consecutive blocks and slides along it, three blocks deep: while block b is searched, block b+1 is
// already normalised, block b+2 is being reduced (tree: 8 samples in the thread, 32 lanes by xor-shuffles,
// warps through shared memory — the same pairs as the definition; one warp then finishes mu, var, r) and
// the loads of block b+3 are in flight; the reduction shares the search's barriers.  z stays in registers;
// widths 1, 2, 4 are formed there from the thread's 8 samples plus 3 of its neighbour's; B_2 is exchanged
// through shared memory for widths 8 and 16, B_4 for width 32, so every level is the definition's own pair
// sum.  Shared arrays are element-major ([element][thread]): every access is conflict free.  Samples at or
// past nout enter as -inf: every window that touches them drops out by itself.
// y is read from HBM once (plus 1/run of halo).  The scan keeps (snr, level, thread) per block — threads own disjoint
// samples, so that already orders the winners; three tiny kernels then count, scan and write the winners that pass
// the threshold, in order, and only there is the sample inside the winning thread's 8 looked up again from y.

#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include <new>

#include "gsp.h"

struct gsp_search {
    int ndm = 0, L = 0, nwidths = 0, device = 0;
    int64_t nout = 0, pitch = 0, max_cand = 0, nblk = 0;
    float threshold = 0.f;
    float *d_best_snr = nullptr;     // [ndm][nblk]
    int32_t *d_best_code = nullptr;  // [ndm][nblk]  (j << 16) | (first sample of the winning thread's 8 - block start)
    float2 *d_blk_stats = nullptr;   // [ndm][nblk]  (mu_f, r_f) of every block
    int32_t *d_row_count = nullptr;  // [ndm]
    int64_t *d_row_off = nullptr;    // [ndm]
};

namespace {

constexpr int kRun = 16;            // blocks per CTA run (halo re-read and pipeline fill: 1/16 of the run)
__constant__ float c_box_scale[6] = {1.0f, 0.70710678f, 0.5f, 0.35355339f, 0.25f, 0.17677669f};

struct Best {
    float snr;
    int code;
};

__device__ __forceinline__ bool better(float s, int c, float bs, int bc) { return s > bs || (s == bs && c < bc); }

// One level of the scan, branch free: the level's eight values are reduced with max, the maximum is scaled
// (x -> fl(x * c_j), c_j > 0, is monotone, so the scaled maximum IS the maximum of the scaled values) and
// kept with its level when it beats the running best (strict '>': an earlier level keeps a tie).  WHICH of
// the eight samples attains it is not tracked here: threads own disjoint sample ranges, so (snr, level,
// thread) already orders any two threads' winners, and the sample inside the winning thread's range is
// looked up only for the winners that become candidates (search_write_kernel).
#define GSP_SCAN_LEVEL(ARR, J)                                                              \
    {                                                                                       \
        const float mr = fmaxf(fmaxf(fmaxf(ARR[0], ARR[1]), fmaxf(ARR[2], ARR[3])),         \
                               fmaxf(fmaxf(ARR[4], ARR[5]), fmaxf(ARR[6], ARR[7])));        \
        const float m = __fmul_rn(mr, c_box_scale[J]);                                      \
        const bool up = m > best.snr;                                                       \
        best.snr = up ? m : best.snr;                                                       \
        best.code = up ? (((J) << 16) | u_loc) : best.code;                                 \
    }

// Everything a thread exchanges with its neighbours is laid out element-major ([element][thread]): lanes then
// touch consecutive words — conflict free — although every thread owns 8 consecutive samples.
template <int NT>
struct SearchSmem {
    float zh[4][3][NT];          // the first three RAW samples of every thread, blocks b .. b + 2 (slot = block & 3)
    float b2s[8][NT + 4];        // B_2 of block b and of the first 32 samples after it
    float b4s[8][NT + 2];        // B_4 likewise (16 samples after it)
    double red[2][8];            // [S1 | S2][warp] of the block being reduced
    float2 sh_stat;              // its statistics, from the warp that finished them
    Best wbest[8];
};

// INTERIOR: every sample the run touches (its blocks and the halo block after them) lies inside the row, so the
// bounds checks of the loads and of the normalisation drop out (all runs of a row but the last one or two).
template <int L, bool INTERIOR>
__device__ __forceinline__ void
search_run(const float *__restrict__ y, int64_t pitch, int64_t nout_, int64_t nblk_, int nwidths,
           float *__restrict__ best_snr, int32_t *__restrict__ best_code, float2 *__restrict__ blk_stats,
           float *__restrict__ stats, SearchSmem<L / 8> &sm) {
    constexpr int NT = L / 8, NW = NT / 32 > 0 ? NT / 32 : 1;
    auto &zh = sm.zh;
    auto &b2s = sm.b2s;
    auto &b4s = sm.b4s;
    auto &red = sm.red;
    float2 &sh_stat = sm.sh_stat;
    auto &wbest = sm.wbest;

    // nout <= 2^31 - 1 (gsp_search_create): block indices and in-row sample indices are 32-bit here
    const int d = blockIdx.y;
    const int nblk = (int)nblk_;
    const unsigned nout = (unsigned)nout_;
    const unsigned rowlen = (unsigned)(pitch < (int64_t)0xffffffffu ? pitch : (int64_t)0xffffffffu);
    const int b_first = (int)blockIdx.x * kRun;
    const int b_last = min(b_first + kRun, nblk);        // exclusive
    const float *row = y + (int64_t)d * pitch;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;

    // The eight samples of block b this thread owns (0 past nout; blocks past the row are not read at all).
    auto load_block = [&](int b, float (&v)[8]) {
        const unsigned u0 = (unsigned)b * L + 8u * t;
        if (INTERIOR ? b < nblk : (b < nblk && u0 + 8u <= nout && u0 + 8u <= rowlen)) {
            const float4 a = __ldg((const float4 *)(row + u0)), c = __ldg((const float4 *)(row + u0 + 4));
            v[0] = a.x, v[1] = a.y, v[2] = a.z, v[3] = a.w, v[4] = c.x, v[5] = c.y, v[6] = c.z, v[7] = c.w;
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = (b < nblk && u0 + i < nout) ? __ldg(row + u0 + i) : 0.f;
        }
    };

    // z of the sample at row index u (raw value yv) with block statistics st; -inf at and past nout
    auto znorm = [&](float yv, unsigned u, float2 st) {
        return (INTERIOR || u < nout) ? __fmul_rn(__fsub_rn(yv, st.x), st.y) : -CUDART_INF_F;
    };

    // First half of staging block b (raw samples in v): the thread's part of the two tree sums goes to red[],
    // its first three RAW samples to zh (the previous thread's boxcars reach into them and normalise them
    // themselves).  The caller's barrier publishes both.
    auto reduce_block = [&](int b, const float (&v)[8]) {
#pragma unroll
        for (int c = 0; c < 3; ++c) zh[b & 3][c][t] = v[c];
        if (b >= nblk) return;
        double p[8], q[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            p[i] = (double)v[i];
            q[i] = __dmul_rn(p[i], p[i]);
        }
        const double s1 = __dadd_rn(__dadd_rn(__dadd_rn(p[0], p[1]), __dadd_rn(p[2], p[3])),
                                    __dadd_rn(__dadd_rn(p[4], p[5]), __dadd_rn(p[6], p[7])));
        const double s2 = __dadd_rn(__dadd_rn(__dadd_rn(q[0], q[1]), __dadd_rn(q[2], q[3])),
                                    __dadd_rn(__dadd_rn(q[4], q[5]), __dadd_rn(q[6], q[7])));
        // both sums in ONE butterfly: at the first level the even lane of a pair takes over the pair's S1,
        // the odd lane its S2 (each sends the other's half), and the remaining four levels run on the
        // lanes of equal parity — the same pairs of the tree, half the shuffles
        const bool odd = (lane & 1) != 0;
        const double send = odd ? s1 : s2, keep = odd ? s2 : s1;
        double acc = __dadd_rn(keep, __shfl_xor_sync(0xffffffffu, send, 1));
#pragma unroll
        for (int o = 2; o < 32; o <<= 1) acc = __dadd_rn(acc, __shfl_xor_sync(0xffffffffu, acc, o));
        if (lane < 2) red[lane][warp] = acc;                // lane 0: S1 of the warp, lane 1: S2
    };
    // Second half, after the barrier that published red[]: the statistics of block b — the tree over the warps,
    // then mu, var, r — computed by the calling warp (every lane the same value).
    auto block_stats = [&](int b) -> float2 {
        if (b >= nblk) return make_float2(0.f, 0.f);
        double a1[8], a2[8];
#pragma unroll
        for (int w = 0; w < NW; ++w) a1[w] = red[0][w], a2[w] = red[1][w];
#pragma unroll
        for (int m = 1; m < NW; m <<= 1)
#pragma unroll
            for (int w = 0; w + m < NW; w += 2 * m) {
                a1[w] = __dadd_rn(a1[w], a1[w + m]);
                a2[w] = __dadd_rn(a2[w], a2[w + m]);
            }
        const unsigned nleft = nout - (unsigned)b * L;
        double mu, m2;
        if (INTERIOR || nleft >= L) {                     // n = L = 2^k: the division is an exact scaling
            mu = __dmul_rn(a1[0], 1.0 / L);
            m2 = __dmul_rn(a2[0], 1.0 / L);
        } else {
            mu = a1[0] / (double)nleft;
            m2 = a2[0] / (double)nleft;
        }
        const double var = __dsub_rn(m2, __dmul_rn(mu, mu));
        const double r = var > 0.0 ? 1.0 / sqrt(var) : 0.0;
        const float2 st = make_float2((float)mu, (float)r);
        if (t == 0) {
            blk_stats[(int64_t)d * nblk + b] = st;
            if (stats) {
                stats[((int64_t)d * nblk + b) * 2] = st.x;
                stats[((int64_t)d * nblk + b) * 2 + 1] = st.y;
            }
        }
        return st;
    };
    // raw samples of block b -> z, in place
    auto normalize_block = [&](int b, float (&v)[8], float2 st) {
        const unsigned u0 = (unsigned)b * L + 8u * t;
        if (b >= nblk) {
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = -CUDART_INF_F;
        } else if (INTERIOR || (unsigned)(b + 1) * L <= nout) {     // CTA-uniform: the whole block is inside the row
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = __fmul_rn(__fsub_rn(v[i], st.x), st.y);
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = znorm(v[i], u0 + i, st);
        }
    };

    // B_1 and B_2 of this thread's eight samples of block `bb` (z in z8) — the three samples after them are
    // the next thread's (same block, statistics st_bb) or thread 0's of the following block (st_nx)
    auto levels012 = [&](int bb, const float (&z8)[8], float2 st_bb, float2 st_nx, float (&b1)[8], float (&b2)[8]) {
        float zz[11];
#pragma unroll
        for (int i = 0; i < 8; ++i) zz[i] = z8[i];
        const bool same = t + 1 < NT;
        const float *h = same ? &zh[bb & 3][0][t + 1] : &zh[(bb + 1) & 3][0][0];
        const unsigned uh = same ? (unsigned)bb * L + 8u * (t + 1) : (unsigned)(bb + 1) * L;
        const float2 sth = same ? st_bb : st_nx;
#pragma unroll
        for (int c = 0; c < 3; ++c) zz[8 + c] = znorm(h[c * NT], uh + c, sth);
        float t1[10];
#pragma unroll
        for (int i = 0; i < 10; ++i) t1[i] = __fadd_rn(zz[i], zz[i + 1]);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            b1[i] = t1[i];
            b2[i] = __fadd_rn(t1[i], t1[i + 2]);
        }
    };
    // B_3[i] = B_2[i] + B_2[i + 4] for 16 samples from this thread's first on, B_4[i] = B_3[i] + B_3[i + 8];
    // `col` = this thread's column of b2s (NT + t for the samples after the block)
    auto levels34 = [&](int col, const float (&own)[8], float (&b3)[8], float (&b4)[8]) {
        float w2[20];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            w2[i] = own[i];
            w2[8 + i] = b2s[i][col + 1];
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) w2[16 + i] = b2s[i][col + 2];
        float t3[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) t3[i] = __fadd_rn(w2[i], w2[i + 4]);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            b3[i] = t3[i];
            b4[i] = __fadd_rn(t3[i], t3[i + 8]);
        }
    };

    // Software pipeline over the blocks of the run, three blocks deep: while block b is searched, block b + 1
    // is already normalised (its first samples are block b's halo), block b + 2 is being reduced — its binary64
    // chain (tree, sqrt, reciprocal) has a whole iteration of float32 search work to hide behind and shares
    // the search's barriers — and the loads of block b + 3 are in flight.  z stays in registers.
    // Blocks past the run's halo block (b_last) are never read: they enter as "absent" (index nblk).
    float zc[8], zn[8], zr[8], v_pre[8];
    load_block(b_first, zc);
    reduce_block(b_first, zc);
    load_block(b_first + 1, zn);
    load_block(b_first + 2 <= b_last ? b_first + 2 : nblk, zr);
    __syncthreads();
    float2 st_c = block_stats(b_first), st_n;
    normalize_block(b_first, zc, st_c);
    __syncthreads();
    reduce_block(b_first + 1, zn);
    __syncthreads();
    st_n = block_stats(b_first + 1);
    normalize_block(b_first + 1, zn, st_n);
    __syncthreads();
    for (int b = b_first; b < b_last; ++b) {
        load_block(b + 3 <= b_last ? b + 3 : nblk, v_pre);
        const bool have2 = b + 2 <= b_last;
        if (have2) reduce_block(b + 2, zr);               // (CTA-uniform) published by the barrier after level 2

        const int u_loc = 8 * t;
        Best best;
        best.snr = -CUDART_INF_F;
        best.code = u_loc;
        float b1[8], b2[8];
        levels012(b, zc, st_c, st_n, b1, b2);
        GSP_SCAN_LEVEL(zc, 0)
        if (nwidths > 1) GSP_SCAN_LEVEL(b1, 1)
        if (nwidths > 2) GSP_SCAN_LEVEL(b2, 2)
        if (nwidths > 3) {                                // uniform over the CTA
#pragma unroll
            for (int i = 0; i < 8; ++i) b2s[i][t] = b2[i];
            float e2[8];
            if (t < 4) {                                  // B_2 of the 32 samples after the block
                float e1[8];
                levels012(b + 1, zn, st_n, st_n, e1, e2);
#pragma unroll
                for (int i = 0; i < 8; ++i) b2s[i][NT + t] = e2[i];
            }
            __syncthreads();
            if (have2 && warp == 0) {                     // one warp finishes block b + 2's statistics
                const float2 st = block_stats(b + 2);
                if (lane == 0) sh_stat = st;
            }
            float b3[8], b4[8];
            levels34(t, b2, b3, b4);
            GSP_SCAN_LEVEL(b3, 3)
            if (nwidths > 4) GSP_SCAN_LEVEL(b4, 4)
            if (nwidths > 5) {
#pragma unroll
                for (int i = 0; i < 8; ++i) b4s[i][t] = b4[i];
                if (t < 2) {                              // B_4 of the 16 samples after the block
                    float e3[8], e4[8];
                    levels34(NT + t, e2, e3, e4);
#pragma unroll
                    for (int i = 0; i < 8; ++i) b4s[i][NT + t] = e4[i];
                }
                __syncthreads();
                float b5[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) b5[i] = __fadd_rn(b4[i], b4s[i][t + 2]);
                GSP_SCAN_LEVEL(b5, 5)
            }
        }

        if (nwidths <= 3) {                               // (no exchange barrier above: publish red[] here)
            __syncthreads();
            if (have2 && warp == 0) {
                const float2 st = block_stats(b + 2);
                if (lane == 0) sh_stat = st;
            }
        }

        // ---- the block's winner: lanes (two warp reductions on order-preserving keys), then warps
        //      (larger snr, then smaller (j, u) code)
        {
            const uint32_t fb = __float_as_uint(best.snr);
            const uint32_t key = (fb & 0x80000000u) ? ~fb : (fb | 0x80000000u);   // monotone in snr
            const uint32_t kmax = __reduce_max_sync(0xffffffffu, key);
            const uint32_t cmin = __reduce_min_sync(0xffffffffu, key == kmax ? (uint32_t)best.code : 0xffffffffu);
            const uint32_t fm = (kmax & 0x80000000u) ? (kmax & 0x7fffffffu) : ~kmax;
            best.snr = __uint_as_float(fm);
            best.code = (int)cmin;
        }
        if (lane == 0) wbest[warp] = best;
        __syncthreads();
        if (t == 0) {
            Best r = wbest[0];
            for (int w = 1; w < NW; ++w)
                if (better(wbest[w].snr, wbest[w].code, r.snr, r.code)) r = wbest[w];
            best_snr[(int64_t)d * nblk + b] = r.snr;
            best_code[(int64_t)d * nblk + b] = r.code;
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            zc[i] = zn[i];
            zn[i] = zr[i];
            zr[i] = v_pre[i];
        }
        st_c = st_n;
        if (have2) {                                      // (after the winner's barrier: sh_stat is published)
            st_n = sh_stat;
            normalize_block(b + 2, zn, st_n);
        }
    }
}

template <int L>
__global__ void __launch_bounds__(L / 8, 768 / (L / 8))
search_blocks_kernel(const float *__restrict__ y, int64_t pitch, int64_t nout, int64_t nblk, int nwidths,
                     float *__restrict__ best_snr, int32_t *__restrict__ best_code, float2 *__restrict__ blk_stats,
                     float *__restrict__ stats) {
    // the run's blocks are [x * kRun, min(., nblk)) and it reads one halo block more: interior when that block ends
    // inside the row (CTA-uniform)
    __shared__ SearchSmem<L / 8> sm;
    const int64_t b_halo_end = ((int64_t)blockIdx.x * kRun + kRun + 1) * L;
    if (b_halo_end <= nout && b_halo_end <= pitch)
        search_run<L, true>(y, pitch, nout, nblk, nwidths, best_snr, best_code, blk_stats, stats, sm);
    else
        search_run<L, false>(y, pitch, nout, nblk, nwidths, best_snr, best_code, blk_stats, stats, sm);
}

// ---- compaction in (DM, block) order: row counts -> exclusive scan -> ordered write
__global__ void __launch_bounds__(256)
search_count_kernel(const float *__restrict__ best_snr, int64_t nblk, float thr, int32_t *__restrict__ row_count) {
    __shared__ int wsum[8];
    const int d = blockIdx.x;
    int n = 0;
    for (int64_t b = threadIdx.x; b < nblk; b += 256) n += best_snr[(int64_t)d * nblk + b] >= thr ? 1 : 0;
    n = __reduce_add_sync(0xffffffffu, n);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = n;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0;
        for (int w = 0; w < 8; ++w) tot += wsum[w];
        row_count[d] = tot;
    }
}

__global__ void __launch_bounds__(1024)
search_scan_kernel(const int32_t *__restrict__ row_count, int ndm, int64_t *__restrict__ row_off,
                   int64_t *__restrict__ total) {
    __shared__ int64_t wsum[32];
    __shared__ int64_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int d0 = 0; d0 < ndm; d0 += 1024) {
        const int d = d0 + threadIdx.x;
        const int64_t v = d < ndm ? row_count[d] : 0;
        int64_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int64_t n = __shfl_up_sync(0xffffffffu, inc, o);
            if ((threadIdx.x & 31) >= o) inc += n;
        }
        if ((threadIdx.x & 31) == 31) wsum[threadIdx.x >> 5] = inc;
        __syncthreads();
        int64_t wbase = 0;
        for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) wbase += wsum[w];
        if (d < ndm) row_off[d] = carry + wbase + inc - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry += wbase + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = carry;
}

// The sample inside a winner's 8-sample range: the boxcar sums of level j over those 8 start samples are formed
// again from y by the tree of the definition (S3, S4) — same operations, same order as the search kernel — and
// the FIRST sample whose snr equals their maximum is the winner's (S5).  Runs for candidates only.
__device__ int winner_sample(const float *__restrict__ row, int64_t nout, int64_t nblk, int L, int64_t b, int j,
                             int u8, const float2 *__restrict__ st_row) {
    const int64_t u0 = b * L + u8;
    const float2 st0 = st_row[b];
    const float2 st1 = (b + 1 < nblk) ? st_row[b + 1] : make_float2(0.f, 0.f);
    float w[40];
    const int n0 = 8 + (1 << j) - 1;                           // samples the 8 windows cover (<= 39)
    for (int i = 0; i < n0; ++i) {
        const int64_t u = u0 + i;
        const float2 st = (u >= (b + 1) * (int64_t)L) ? st1 : st0;
        w[i] = (u < nout) ? __fmul_rn(__fsub_rn(__ldg(row + u), st.x), st.y) : -CUDART_INF_F;
    }
    int n = n0;
    for (int k = 0; k < j; ++k) {                              // B_{k+1}[i] = B_k[i] + B_k[i + 2^k]
        n -= 1 << k;
        for (int i = 0; i < n; ++i) w[i] = __fadd_rn(w[i], w[i + (1 << k)]);
    }
    const float cj = c_box_scale[j];
    float mx = -CUDART_INF_F;
    int at = 0;
    for (int i = 0; i < 8; ++i) {
        const float v = __fmul_rn(w[i], cj);
        if (v > mx) {
            mx = v;
            at = i;
        }
    }
    return u8 + at;
}

__global__ void __launch_bounds__(256)
search_write_kernel(const float *__restrict__ y, int64_t pitch, int64_t nout, const float *__restrict__ best_snr,
                    const int32_t *__restrict__ best_code, const float2 *__restrict__ blk_stats, int64_t nblk, int L,
                    float thr, const int64_t *__restrict__ row_off, int64_t max_cand, int32_t *__restrict__ c_dm,
                    int32_t *__restrict__ c_u, int32_t *__restrict__ c_w, float *__restrict__ c_snr) {
    __shared__ int wsum[8];
    __shared__ int64_t base;
    const int d = blockIdx.x;
    if (threadIdx.x == 0) base = row_off[d];
    __syncthreads();
    for (int64_t b0 = 0; b0 < nblk; b0 += 256) {
        const int64_t b = b0 + threadIdx.x;
        const float s = b < nblk ? best_snr[(int64_t)d * nblk + b] : -CUDART_INF_F;
        const bool hit = b < nblk && s >= thr;
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        if (lane == 0) wsum[warp] = __popc(m);
        __syncthreads();
        int before = __popc(m & ((1u << lane) - 1u));
        for (int w = 0; w < warp; ++w) before += wsum[w];
        if (hit) {
            const int64_t k = base + before;
            if (k < max_cand) {
                const int code = best_code[(int64_t)d * nblk + b];
                const int j = code >> 16;
                const int u_in = winner_sample(y + (int64_t)d * pitch, nout, nblk, L, b, j, code & 0xffff,
                                               blk_stats + (int64_t)d * nblk);
                c_dm[k] = d;
                c_u[k] = (int32_t)(b * L + u_in);
                c_w[k] = 1 << j;
                c_snr[k] = s;
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int tot = 0;
            for (int w = 0; w < 8; ++w) tot += wsum[w];
            base += tot;
        }
        __syncthreads();
    }
}

}  // namespace

extern "C" {

gsp_status gsp_search_create(gsp_search **out, int ndm, int64_t nout, int64_t pitch, int block, int nwidths,
                             float threshold, int64_t max_cand) {
    if (!out) return GSP_ERR_INVALID_ARG;
    *out = nullptr;
    if (ndm < 1 || ndm > 65535 || nout < 1 || pitch < nout || nwidths < 1 || nwidths > 6 || max_cand < 0)
        return GSP_ERR_INVALID_ARG;
    if (!(block == 256 || block == 512 || block == 1024 || block == 2048)) return GSP_ERR_INVALID_ARG;
    if (!(threshold == threshold) || nout > 0x7fffffff) return GSP_ERR_INVALID_ARG;
    gsp_search *s = new (std::nothrow) gsp_search();
    if (!s) return GSP_ERR_ALLOC;
    s->ndm = ndm;
    s->nout = nout;
    s->pitch = pitch;
    s->L = block;
    s->nwidths = nwidths;
    s->threshold = threshold;
    s->max_cand = max_cand;
    s->nblk = (nout + block - 1) / block;
    cudaError_t e = cudaGetDevice(&s->device);
    const size_t cells = (size_t)ndm * (size_t)s->nblk;
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->d_best_snr, cells * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->d_best_code, cells * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->d_blk_stats, cells * sizeof(float2));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->d_row_count, (size_t)ndm * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->d_row_off, (size_t)ndm * sizeof(int64_t));
    if (e != cudaSuccess) {
        const gsp_status st = (e == cudaErrorMemoryAllocation) ? GSP_ERR_ALLOC : GSP_ERR_CUDA;
        cudaGetLastError();
        gsp_search_destroy(s);
        return st;
    }
    *out = s;
    return GSP_OK;
}

gsp_status gsp_search_run(gsp_search *s, const float *d_y, int32_t *d_cand_dm, int32_t *d_cand_sample,
                          int32_t *d_cand_width, float *d_cand_snr, int64_t *d_count, float *d_stats,
                          void *cuda_stream) {
    if (!s || !d_y || !d_count) return GSP_ERR_INVALID_ARG;
    if (s->max_cand > 0 && (!d_cand_dm || !d_cand_sample || !d_cand_width || !d_cand_snr)) return GSP_ERR_INVALID_ARG;
    if ((uintptr_t)d_y & 15) return GSP_ERR_INVALID_ARG;
    if (s->pitch % 4 != 0 && s->ndm > 1) return GSP_ERR_INVALID_ARG;   // rows must stay 16-byte aligned
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != s->device) return GSP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const dim3 grid((unsigned)((s->nblk + kRun - 1) / kRun), (unsigned)s->ndm);
#define GSP_SEARCH_LAUNCH(LL)                                                                               \
    search_blocks_kernel<LL><<<grid, LL / 8, 0, st>>>(d_y, s->pitch, s->nout, s->nblk, s->nwidths,         \
                                                      s->d_best_snr, s->d_best_code, s->d_blk_stats, d_stats)
    switch (s->L) {
        case 256: GSP_SEARCH_LAUNCH(256); break;
        case 512: GSP_SEARCH_LAUNCH(512); break;
        case 1024: GSP_SEARCH_LAUNCH(1024); break;
        default: GSP_SEARCH_LAUNCH(2048); break;
    }
#undef GSP_SEARCH_LAUNCH
    search_count_kernel<<<s->ndm, 256, 0, st>>>(s->d_best_snr, s->nblk, s->threshold, s->d_row_count);
    search_scan_kernel<<<1, 1024, 0, st>>>(s->d_row_count, s->ndm, s->d_row_off, d_count);
    if (s->max_cand > 0)
        search_write_kernel<<<s->ndm, 256, 0, st>>>(d_y, s->pitch, s->nout, s->d_best_snr, s->d_best_code,
                                                    s->d_blk_stats, s->nblk, s->L, s->threshold, s->d_row_off,
                                                    s->max_cand, d_cand_dm, d_cand_sample, d_cand_width, d_cand_snr);
    if (cudaPeekAtLastError() != cudaSuccess) {
        cudaGetLastError();
        return GSP_ERR_CUDA;
    }
    return GSP_OK;
}

int64_t gsp_search_nblocks(const gsp_search *s) { return s ? s->nblk : 0; }

gsp_status gsp_search_destroy(gsp_search *s) {
    if (!s) return GSP_OK;
    cudaFree(s->d_best_snr);
    cudaFree(s->d_best_code);
    cudaFree(s->d_blk_stats);
    cudaFree(s->d_row_count);
    cudaFree(s->d_row_off);
    cudaGetLastError();
    delete s;
    return GSP_OK;
}

}  // extern "C"
