// gsp_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU statement of two-stage subband incoherent
// dedispersion (PRESTO "prepsubband" as named by the paper, §2.3).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may build, load or call this file.  It shares no code, header,
// table generator or constant with paper_2110_12749_b200/csrc (the CUDA path).
//
// What it follows (P:NNN = line of /root/reference/PAPER.md, BJ = BASELINE.json):
//   * shift-and-sum semantic  result[kk] += data[kk + delay[ii]][ii]
//       — Algorithm 1, P:104-136 (read per SURVEY §8(c) A9: outer loop over DMs,
//         lastdata||data is one contiguous time axis);
//   * one independent sum per (DM, sample)  — Algorithm 2, P:142-166;
//   * matrices numpts x numchan in, numdm x numpts out, float32 out — P:102, P:206;
//   * sub-band method: channels -> subbands at one subband DM, subbands -> trial
//     DMs — P:100 (named only); mechanics from BJ.north_star + SURVEY §8(c) O1-O6;
//   * delay constant and formula  dt = 4.148808e3 s * DM * (f^-2 - fref^-2), MHz
//       — BJ.north_star (the paper is silent, "pre-calculated");
//   * DownSamp between the stages, mean of ds consecutive subband samples
//       — Tables 2-3 P:39-64 (column only), reading A7 in DESIGN.md.
//
// Pins (tests/test_oracle_pins.py, all run with -m "not gpu"): P1 DM=0 plain
// channel sum, P2 one-stage brute force with composite shifts, P3 rounding bound,
// P4 linearity, P5 time-shift equivariance, P6 impulse closed form, P7 constant
// input, P8 ramp closed form, P9 table structure, P10 block-carry concatenation,
// P11 Tiny worked example, P12 table extents.  Agreement with a real PRESTO run:
// PARITY UNPINNED (PRESTO is not available).
//
// Precision: tables in IEEE binary64, rule R3; uint8 input summed in int64 (exact);
// float32 input summed in binary64 and rounded to float32 once at the end.

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// BJ.north_star: "dt = 4.148808e3 s * DM * (f^-2 - f_ref^-2) with MHz inputs".
const double kDispersionConstant = 4.148808e3;

// Rule R3: binary64, operations in the order written, floor(x + 0.5).
long long round_delay(double dm, double f_mhz, double fref_mhz, double tsamp_s) {
    double inv_f2 = 1.0 / (f_mhz * f_mhz);
    double inv_r2 = 1.0 / (fref_mhz * fref_mhz);
    double x = (kDispersionConstant * dm) * (inv_f2 - inv_r2) / tsamp_s;
    return (long long)std::floor(x + 0.5);
}

// O1: centre frequency of channel c; channel 0 is the highest frequency (A2).
double chan_freq(double f_top, double chan_bw, int c) { return f_top + (double)c * chan_bw; }

template <typename T> struct Acc;
template <> struct Acc<uint8_t> { typedef long long type; };
template <> struct Acc<float>   { typedef double type; };

// O4 + O5 for one subband: S_s[t] = sum_{c in s} x[t + s1[c]][c], t in [0, n1);
// S'_s[u] = (1/ds) sum_{k<ds} S_s[u*ds + k], u in [0, n1d).  The 1/ds factor is
// applied at the very end (O6) so that integer sums stay integer: here S' holds
// the un-divided sum over k.
template <typename T>
void stage1_one_subband(const T* x, int nchan, int cps, int s, const int32_t* s1,
                        long long n1d, int ds, typename Acc<T>::type* Sp) {
    typedef typename Acc<T>::type A;
    for (long long u = 0; u < n1d; ++u) {
        A tot = 0;
        for (int k = 0; k < ds; ++k) {
            long long t = u * ds + k;
            for (int j = 0; j < cps; ++j) {
                int c = s * cps + j;
                tot += (A)x[(t + s1[c]) * (long long)nchan + c];
            }
        }
        Sp[u] = tot;
    }
}

template <typename T>
int dedisperse(const T* x, long long nsamp, int nchan, int nsub, const int32_t* s1,
               const int32_t* s2, int ndm, int ds, float* y, long long pitch, int nthreads) {
    typedef typename Acc<T>::type A;
    if (!x || !s1 || !s2 || !y || nchan < 1 || nsub < 1 || nchan % nsub || ndm < 1 || ds < 1)
        return 1;
    const int cps = nchan / nsub;
    long long H1 = 0, H2 = 0;
    for (int c = 0; c < nchan; ++c) if (s1[c] > H1) H1 = s1[c];
    for (long long i = 0; i < (long long)ndm * nsub; ++i) if (s2[i] > H2) H2 = s2[i];
    const long long n1 = nsamp - H1;
    if (n1 <= 0) return 2;
    const long long n1d = n1 / ds;            // trailing n1 mod ds samples dropped (O5)
    const long long nout = n1d - H2;          // valid-only output (A8)
    if (nout <= 0) return 2;
    if (pitch < nout) return 1;
    (void)nthreads;

    std::vector<A> Sp((size_t)nsub * (size_t)n1d);
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (int s = 0; s < nsub; ++s)
        stage1_one_subband<T>(x, nchan, cps, s, s1, n1d, ds, Sp.data() + (size_t)s * n1d);

    // O6: y_d[u] = (1/ds) * sum_s S'_s[u + s2[d][s]].
    const double inv_ds = 1.0 / (double)ds;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (int d = 0; d < ndm; ++d) {
        std::vector<A> row((size_t)nout, (A)0);
        for (int s = 0; s < nsub; ++s) {
            const A* src = Sp.data() + (size_t)s * n1d + s2[(size_t)d * nsub + s];
            for (long long u = 0; u < nout; ++u) row[u] += src[u];
        }
        float* yd = y + (size_t)d * pitch;
        for (long long u = 0; u < nout; ++u) yd[u] = (float)((double)row[u] * inv_ds);
    }
    return 0;
}

// One output sample straight from the definition (O4-O6 written out for a point):
// used at full benchmark sizes where the whole matrix is too slow to compute.
template <typename T>
float one_point(const T* x, int nchan, int nsub, const int32_t* s1, const int32_t* s2,
                int ds, int d, long long u) {
    typedef typename Acc<T>::type A;
    const int cps = nchan / nsub;
    A tot = 0;
    for (int s = 0; s < nsub; ++s) {
        long long v = u + s2[(size_t)d * nsub + s];          // index into S'_s
        for (int k = 0; k < ds; ++k) {
            long long t = v * ds + k;                         // index into S_s
            for (int j = 0; j < cps; ++j) {
                int c = s * cps + j;
                tot += (A)x[(t + s1[c]) * (long long)nchan + c];
            }
        }
    }
    return (float)((double)tot * (1.0 / (double)ds));
}

}  // namespace

extern "C" {

// O1-O3 + rule R3.  s1: nchan entries; s2: ndm*nsub entries, DM-major.
int gsp_oracle_tables(int nchan, double f_top, double chan_bw, double dt, int nsub,
                      double subband_dm, const double* dm_list, int ndm, int ds,
                      int32_t* s1, int32_t* s2) {
    if (nchan < 1 || nsub < 1 || nchan % nsub || ndm < 1 || ds < 1 || !dm_list || !s1 || !s2)
        return 1;
    if (!(chan_bw < 0.0) || !(dt > 0.0)) return 1;
    if (!(chan_freq(f_top, chan_bw, nchan - 1) > 0.0)) return 1;
    const int cps = nchan / nsub;
    const double f0 = chan_freq(f_top, chan_bw, 0);                 // global reference (O1)
    for (int c = 0; c < nchan; ++c) {
        int s = c / cps;
        double fref = chan_freq(f_top, chan_bw, s * cps);           // subband's top channel (A3)
        s1[c] = (int32_t)round_delay(subband_dm, chan_freq(f_top, chan_bw, c), fref, dt);   // R1
    }
    for (int d = 0; d < ndm; ++d)
        for (int s = 0; s < nsub; ++s) {
            double fref = chan_freq(f_top, chan_bw, s * cps);
            s2[(size_t)d * nsub + s] =
                (int32_t)round_delay(dm_list[d], fref, f0, dt * (double)ds);                // R2
        }
    return 0;
}

int gsp_oracle_dedisperse_u8(const uint8_t* x, long long nsamp, int nchan, int nsub,
                             const int32_t* s1, const int32_t* s2, int ndm, int ds,
                             float* y, long long pitch, int nthreads) {
    return dedisperse<uint8_t>(x, nsamp, nchan, nsub, s1, s2, ndm, ds, y, pitch, nthreads);
}

int gsp_oracle_dedisperse_f32(const float* x, long long nsamp, int nchan, int nsub,
                              const int32_t* s1, const int32_t* s2, int ndm, int ds,
                              float* y, long long pitch, int nthreads) {
    return dedisperse<float>(x, nsamp, nchan, nsub, s1, s2, ndm, ds, y, pitch, nthreads);
}

int gsp_oracle_points_u8(const uint8_t* x, int nchan, int nsub, const int32_t* s1,
                         const int32_t* s2, int ds, const int32_t* d_idx,
                         const long long* u_idx, long long npts, float* out) {
    for (long long i = 0; i < npts; ++i)
        out[i] = one_point<uint8_t>(x, nchan, nsub, s1, s2, ds, d_idx[i], u_idx[i]);
    return 0;
}

int gsp_oracle_points_f32(const float* x, int nchan, int nsub, const int32_t* s1,
                          const int32_t* s2, int ds, const int32_t* d_idx,
                          const long long* u_idx, long long npts, float* out) {
    for (long long i = 0; i < npts; ++i)
        out[i] = one_point<float>(x, nchan, nsub, s1, s2, ds, d_idx[i], u_idx[i]);
    return 0;
}

int gsp_oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
