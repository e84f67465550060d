// gsp_extras_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain CPU statements of the two steps of the GSP pipeline that sit directly before and after
// the dedispersion path:
//
//   * the RFI prologue applied to the filterbank before dedispersion — "pulsar search (RFI
//     mitigation, de-dispersion and single-pulse search)" PAPER.md:82, the 'mask' and 'clip'
//     options of prepsubband PAPER.md:208;
//   * the single-pulse search applied to every dedispersed time series — PAPER.md:82, :86
//     ("the single-pulse search ... parallel executed on CPU").
//
// The paper names these steps and gives NO mechanics for either (no formula, threshold, width set
// or statistic is printed anywhere in PAPER.md).  What is computed here is therefore the set of
// readings F1-F4 / S1-S6 listed in DESIGN.md §3a, written out step by step; every floating-point
// decision is taken in a stated precision and a stated order so that the CUDA path can take the
// same decision bit for bit.  Shares no code with paper_2110_12749_b200/csrc.  Compiled with
// -ffp-contract=off: no fused multiply-add anywhere.
//
// Pins: tests/test_extras_pins.py (all -m "not gpu").  Agreement with PRESTO's rfifind / clip /
// single_pulse_search.py: PARITY UNPINNED (PRESTO is not available, and the paper does not say
// which of their parameters GSP used).

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <vector>

namespace {

// ------------------------------------------------------------------------------------------
// RFI prologue (uint8 filterbank, the paper's 8-bit data PAPER.md:176)
// ------------------------------------------------------------------------------------------
// F1 channel mask  x1[t][c] = mask[c] ? pad[c] : x[t][c]
// F2 zero-DM       z[t] = sum_c x1[t][c]                         (exact integer)
// F3 clip          per block of B rows (last block ragged, n rows): S1 = sum z, S2 = sum z^2;
//                  row t is clipped iff  (double)(n*z[t] - S1) > clip_sigma * sqrt((double)(n*S2 - S1*S1))
//                  i.e. z[t] - mean > clip_sigma * std, all integer parts exact in int64
//                  (requires B * nchan * 255 < 2^31), one sqrt and one product in binary64
// F4 replace       x2[t][c] = clipped[t] ? pad[c] : x1[t][c]
int rfi_prologue(const uint8_t* x, long long nsamp, int nchan, const uint8_t* mask,
                 const uint8_t* pad, double clip_sigma, int clip_block, uint8_t* x2,
                 long long* z_out, uint8_t* clipped_out) {
    if (!x || !pad || !x2 || nsamp < 1 || nchan < 1) return 1;
    if (clip_sigma > 0.0 && (clip_block < 2 || (long long)clip_block * nchan * 255 >= (1LL << 31))) return 1;
    std::vector<long long> z((size_t)nsamp, 0);
    for (long long t = 0; t < nsamp; ++t) {
        long long tot = 0;
        for (int c = 0; c < nchan; ++c) {
            uint8_t v = (mask && mask[c]) ? pad[c] : x[t * (long long)nchan + c];      // F1
            x2[t * (long long)nchan + c] = v;
            tot += v;                                                                   // F2
        }
        z[(size_t)t] = tot;
        if (z_out) z_out[t] = tot;
        if (clipped_out) clipped_out[t] = 0;
    }
    if (!(clip_sigma > 0.0)) return 0;
    for (long long t0 = 0; t0 < nsamp; t0 += clip_block) {                              // F3
        long long n = nsamp - t0 < clip_block ? nsamp - t0 : clip_block;
        long long S1 = 0, S2 = 0;
        for (long long t = t0; t < t0 + n; ++t) {
            S1 += z[(size_t)t];
            S2 += z[(size_t)t] * z[(size_t)t];
        }
        double rhs = clip_sigma * std::sqrt((double)(n * S2 - S1 * S1));
        for (long long t = t0; t < t0 + n; ++t) {
            if ((double)(n * z[(size_t)t] - S1) > rhs) {
                if (clipped_out) clipped_out[t] = 1;
                for (int c = 0; c < nchan; ++c) x2[t * (long long)nchan + c] = pad[c];  // F4
            }
        }
    }
    return 0;
}

// ------------------------------------------------------------------------------------------
// single-pulse search on dedispersed series y[ndm][pitch] (float32), nout valid samples per row
// ------------------------------------------------------------------------------------------
// S1 blocks of L = 2^k samples (last block ragged, n samples).  Block sums S1 = sum y, S2 = sum y*y
//    in binary64, added in a PERFECT BINARY TREE over the L slots of the block in natural order
//    (absent slots of a ragged block count as 0): tree(a, lo, len) = tree(lo, len/2) + tree(lo+len/2, len/2).
// S2 mu = S1/n; var = S2/n - mu*mu (separate multiply and subtract); var <= 0 -> r = 0 else
//    r = 1/sqrt(var); mu_f = (float)mu, r_f = (float)r.
// S3 z[u] = (y[u] - mu_f) * r_f in float32 (each sample with the statistics of its own block).
// S4 boxcars of widths 2^j: B_0 = z, B_{j+1}[u] = B_j[u] + B_j[u + 2^j] (float32), defined while
//    u + 2^(j+1) <= nout; snr_j[u] = B_j[u] * c_j with c_j = 2^(-j/2) as the float32 constants below.
// S5 per (DM d, block b): the best (snr, j, u) over u in the block and j < nwidths with u + 2^j <= nout,
//    ordered by larger snr, then smaller j, then smaller u.
// S6 it is a candidate iff snr >= threshold; candidates are listed in (d, b) order.
const float kBoxScale[8] = {1.0f, 0.70710678f, 0.5f, 0.35355339f, 0.25f, 0.17677669f, 0.125f, 0.088388348f};

double tree_sum(const double* a, long long len) {
    if (len == 1) return a[0];
    return tree_sum(a, len / 2) + tree_sum(a + len / 2, len / 2);
}

long long search(const float* y, int ndm, long long nout, long long pitch, int L, int nwidths,
                 float threshold, long long max_cand, int32_t* c_dm, int32_t* c_u, int32_t* c_w,
                 float* c_snr, float* stats /* optional [ndm][nblk][2] mu_f, r_f */) {
    if (!y || ndm < 1 || nout < 1 || pitch < nout || L < 2 || (L & (L - 1)) || nwidths < 1 || nwidths > 8)
        return -1;
    const long long nblk = (nout + L - 1) / L;
    long long count = 0;
    std::vector<float> z((size_t)nout), B((size_t)nout), Bn((size_t)nout);
    std::vector<double> v1((size_t)L), v2((size_t)L);
    std::vector<float> best_snr((size_t)nblk);
    std::vector<int> best_j((size_t)nblk);
    std::vector<long long> best_u((size_t)nblk);
    for (int d = 0; d < ndm; ++d) {
        const float* row = y + (size_t)d * pitch;
        for (long long b = 0; b < nblk; ++b) {                                  // S1-S3
            long long u0 = b * L, n = nout - u0 < L ? nout - u0 : L;
            for (long long i = 0; i < L; ++i) {
                double v = i < n ? (double)row[u0 + i] : 0.0;
                v1[(size_t)i] = v;
                v2[(size_t)i] = v * v;
            }
            double S1 = tree_sum(v1.data(), L), S2 = tree_sum(v2.data(), L);
            double mu = S1 / (double)n;
            double musq = mu * mu;
            double var = S2 / (double)n - musq;
            double r = var > 0.0 ? 1.0 / std::sqrt(var) : 0.0;
            float mu_f = (float)mu, r_f = (float)r;
            if (stats) {
                stats[((size_t)d * nblk + b) * 2] = mu_f;
                stats[((size_t)d * nblk + b) * 2 + 1] = r_f;
            }
            for (long long i = 0; i < n; ++i) {
                float dlt = row[u0 + i] - mu_f;
                z[(size_t)(u0 + i)] = dlt * r_f;
            }
            best_snr[(size_t)b] = -INFINITY;
            best_j[(size_t)b] = 0;
            best_u[(size_t)b] = u0;
        }
        B = z;
        for (int j = 0; j < nwidths; ++j) {                                     // S4, S5
            long long w = 1LL << j;
            if (w > nout) break;
            long long nvalid = nout - w + 1;                                    // u + 2^j <= nout
            for (long long u = 0; u < nvalid; ++u) {
                float snr = B[(size_t)u] * kBoxScale[j];
                long long b = u / L;
                if (snr > best_snr[(size_t)b]) {        // strict: ties keep the smaller j, then the smaller u
                    best_snr[(size_t)b] = snr;
                    best_j[(size_t)b] = j;
                    best_u[(size_t)b] = u;
                }
            }
            if (j + 1 < nwidths && 2 * w <= nout) {
                long long nnext = nout - 2 * w + 1;
                for (long long u = 0; u < nnext; ++u) Bn[(size_t)u] = B[(size_t)u] + B[(size_t)(u + w)];
                B.swap(Bn);
            }
        }
        for (long long b = 0; b < nblk; ++b) {                                  // S6
            if (best_snr[(size_t)b] >= threshold) {
                if (count < max_cand) {
                    c_dm[count] = d;
                    c_u[count] = (int32_t)best_u[(size_t)b];
                    c_w[count] = 1 << best_j[(size_t)b];
                    c_snr[count] = best_snr[(size_t)b];
                }
                ++count;
            }
        }
    }
    return count;
}

}  // namespace

extern "C" {

int gsp_oracle_rfi_prologue(const uint8_t* x, long long nsamp, int nchan, const uint8_t* mask,
                            const uint8_t* pad, double clip_sigma, int clip_block, uint8_t* x2,
                            long long* z_out, uint8_t* clipped_out) {
    return rfi_prologue(x, nsamp, nchan, mask, pad, clip_sigma, clip_block, x2, z_out, clipped_out);
}

long long gsp_oracle_search(const float* y, int ndm, long long nout, long long pitch, int L,
                            int nwidths, float threshold, long long max_cand, int32_t* c_dm,
                            int32_t* c_u, int32_t* c_w, float* c_snr, float* stats) {
    return search(y, ndm, nout, pitch, L, nwidths, threshold, max_cand, c_dm, c_u, c_w, c_snr, stats);
}

}  // extern "C"
