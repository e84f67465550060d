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
// of consecutive blocks and slides along it: while block b is searched, block b+1 has already been loaded,
// reduced (tree: 8 samples in the thread, 32 lanes by xor-shuffles, warps through shared memory — the same
// pairs as the definition) and normalised into the other half of a 2L-sample shared buffer, which supplies
// the 31-sample halo the boxcars need.  Widths 1, 2, 4 are formed in registers from 11 loaded samples; B_2
// is staged in shared memory for widths 8 and 16, B_4 for width 32, so every level is the definition's own
// pair sum.  Samples at or past nout enter as -inf: every window that touches them drops out by itself.
// y is read from HBM once (plus 1/run of halo); a second tiny kernel pair compacts the per-(DM, block)
// winners that pass the threshold into the candidate list, in order.

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
    int32_t *d_best_code = nullptr;  // [ndm][nblk]  (j << 16) | (u - block start)
    int32_t *d_row_count = nullptr;  // [ndm]
    int64_t *d_row_off = nullptr;    // [ndm]
};

namespace {

constexpr int kRun = 16;            // blocks per CTA run (halo re-read: 1/16 of a block per run)
__constant__ float c_box_scale[6] = {1.0f, 0.70710678f, 0.5f, 0.35355339f, 0.25f, 0.17677669f};

struct Best {
    float snr;
    int code;
};

__device__ __forceinline__ bool better(float s, int c, float bs, int bc) { return s > bs || (s == bs && c < bc); }

// One level of the scan: samples in ascending order, strict '>' keeps the earliest of equal values.
#define GSP_SCAN_LEVEL(ARR, J)                                           \
    {                                                                    \
        const float cj = c_box_scale[J];                                 \
        _Pragma("unroll") for (int i = 0; i < 8; ++i) {                  \
            const float s = __fmul_rn(ARR[i], cj);                       \
            if (s > best.snr) {                                          \
                best.snr = s;                                            \
                best.code = ((J) << 16) | (u_loc + i);                   \
            }                                                            \
        }                                                                \
    }

template <int L>
__global__ void __launch_bounds__(L / 8)
search_blocks_kernel(const float *__restrict__ y, int64_t pitch, int64_t nout, int64_t nblk, int nwidths,
                     float *__restrict__ best_snr, int32_t *__restrict__ best_code, float *__restrict__ stats) {
    constexpr int NT = L / 8, NW = NT / 32 > 0 ? NT / 32 : 1;
    __shared__ __align__(16) float zbuf[2 * L];          // block b at (b & 1) * L, block b + 1 in the other half
    __shared__ __align__(16) float b2s[L + 32];          // B_2 of block b and of the first 32 samples after it
    __shared__ __align__(16) float b4s[L + 16];          // B_4 likewise (16 samples after it)
    __shared__ double red[2][8];
    __shared__ float2 sh_stat;
    __shared__ Best wbest[8];

    const int d = blockIdx.y;
    const int64_t b_first = (int64_t)blockIdx.x * kRun;
    const int64_t b_last = min(b_first + kRun, nblk);    // exclusive
    const float *row = y + (int64_t)d * pitch;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;

    // Load block b, reduce, normalise into its half of zbuf.  Blocks past the row are all -inf.
    auto stage_block = [&](int64_t b) {
        float *zdst = zbuf + (b & 1) * L + 8 * t;
        const int64_t u0 = b * L + 8 * t;
        float v[8];
        if (b < nblk) {
            if (u0 + 8 <= nout && u0 + 8 <= pitch) {
                const float4 a = __ldg((const float4 *)(row + u0)), c = __ldg((const float4 *)(row + u0 + 4));
                v[0] = a.x, v[1] = a.y, v[2] = a.z, v[3] = a.w, v[4] = c.x, v[5] = c.y, v[6] = c.z, v[7] = c.w;
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) v[i] = (u0 + i < nout) ? __ldg(row + u0 + i) : 0.f;
            }
            double p[8], q[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                p[i] = (double)v[i];
                q[i] = __dmul_rn(p[i], p[i]);
            }
            double s1 = __dadd_rn(__dadd_rn(__dadd_rn(p[0], p[1]), __dadd_rn(p[2], p[3])),
                                  __dadd_rn(__dadd_rn(p[4], p[5]), __dadd_rn(p[6], p[7])));
            double s2 = __dadd_rn(__dadd_rn(__dadd_rn(q[0], q[1]), __dadd_rn(q[2], q[3])),
                                  __dadd_rn(__dadd_rn(q[4], q[5]), __dadd_rn(q[6], q[7])));
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                s1 = __dadd_rn(s1, __shfl_xor_sync(0xffffffffu, s1, o));
                s2 = __dadd_rn(s2, __shfl_xor_sync(0xffffffffu, s2, o));
            }
            if (lane == 0) {
                red[0][warp] = s1;
                red[1][warp] = s2;
            }
            __syncthreads();
            if (t == 0) {
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
                const int64_t nleft = nout - b * L;
                const double n = (double)(nleft < L ? nleft : L);
                const double mu = a1[0] / n;
                const double var = __dsub_rn(a2[0] / n, __dmul_rn(mu, mu));
                const double r = var > 0.0 ? 1.0 / sqrt(var) : 0.0;
                sh_stat = make_float2((float)mu, (float)r);
                if (stats) {
                    stats[((int64_t)d * nblk + b) * 2] = (float)mu;
                    stats[((int64_t)d * nblk + b) * 2 + 1] = (float)r;
                }
            }
            __syncthreads();
            const float2 st = sh_stat;
#pragma unroll
            for (int i = 0; i < 8; ++i)
                v[i] = (u0 + i < nout) ? __fmul_rn(__fsub_rn(v[i], st.x), st.y) : -CUDART_INF_F;
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = -CUDART_INF_F;
        }
        *(float4 *)zdst = make_float4(v[0], v[1], v[2], v[3]);
        *(float4 *)(zdst + 4) = make_float4(v[4], v[5], v[6], v[7]);
    };

    // B_1 and B_2 of the eight samples starting at ring position `pos` (a multiple of 8) of zbuf
    auto levels012 = [&](int pos, float (&z8)[8], float (&b1)[8], float (&b2)[8]) {
        float zz[11];
        const float4 a = *(const float4 *)(zbuf + pos), c = *(const float4 *)(zbuf + pos + 4);
        zz[0] = a.x, zz[1] = a.y, zz[2] = a.z, zz[3] = a.w, zz[4] = c.x, zz[5] = c.y, zz[6] = c.z, zz[7] = c.w;
#pragma unroll
        for (int i = 8; i < 11; ++i) zz[i] = zbuf[(pos + i) & (2 * L - 1)];
        float t1[10];
#pragma unroll
        for (int i = 0; i < 10; ++i) t1[i] = __fadd_rn(zz[i], zz[i + 1]);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            z8[i] = zz[i];
            b1[i] = t1[i];
            b2[i] = __fadd_rn(t1[i], t1[i + 2]);
        }
    };

    stage_block(b_first);
    for (int64_t b = b_first; b < b_last; ++b) {
        stage_block(b + 1);                               // (its internal barriers also order the reuse of zbuf)
        __syncthreads();

        const int base = (int)(b & 1) * L;                // ring position of this block
        const int u_loc = 8 * t;
        Best best;
        best.snr = -CUDART_INF_F;
        best.code = u_loc;
        float z8[8], b1[8], b2[8];
        levels012(base + u_loc, z8, b1, b2);
        GSP_SCAN_LEVEL(z8, 0)
        if (nwidths > 1) GSP_SCAN_LEVEL(b1, 1)
        if (nwidths > 2) GSP_SCAN_LEVEL(b2, 2)
        if (nwidths > 3) {                                // uniform over the CTA
            *(float4 *)(b2s + u_loc) = make_float4(b2[0], b2[1], b2[2], b2[3]);
            *(float4 *)(b2s + u_loc + 4) = make_float4(b2[4], b2[5], b2[6], b2[7]);
            if (t < 4) {                                  // B_2 of the 32 samples after the block
                float e0[8], e1[8], e2[8];
                levels012((base + L + u_loc) & (2 * L - 1), e0, e1, e2);
                *(float4 *)(b2s + L + u_loc) = make_float4(e2[0], e2[1], e2[2], e2[3]);
                *(float4 *)(b2s + L + u_loc + 4) = make_float4(e2[4], e2[5], e2[6], e2[7]);
            }
            __syncthreads();
            // B_3[i] = B_2[i] + B_2[i + 4] for the 16 samples from u_loc on; B_4[i] = B_3[i] + B_3[i + 8]
            auto levels34 = [&](int p, float (&b3)[8], float (&b4)[8]) {
                float w2[20];
#pragma unroll
                for (int k = 0; k < 5; ++k) {
                    const float4 a = *(const float4 *)(b2s + p + 4 * k);
                    w2[4 * k] = a.x, w2[4 * k + 1] = a.y, w2[4 * k + 2] = a.z, w2[4 * k + 3] = a.w;
                }
                float t3[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) t3[i] = __fadd_rn(w2[i], w2[i + 4]);
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    b3[i] = t3[i];
                    b4[i] = __fadd_rn(t3[i], t3[i + 8]);
                }
            };
            float b3[8], b4[8];
            levels34(u_loc, b3, b4);
            GSP_SCAN_LEVEL(b3, 3)
            if (nwidths > 4) GSP_SCAN_LEVEL(b4, 4)
            if (nwidths > 5) {
                *(float4 *)(b4s + u_loc) = make_float4(b4[0], b4[1], b4[2], b4[3]);
                *(float4 *)(b4s + u_loc + 4) = make_float4(b4[4], b4[5], b4[6], b4[7]);
                if (t < 2) {                              // B_4 of the 16 samples after the block
                    float e3[8], e4[8];
                    levels34(L + u_loc, e3, e4);
                    *(float4 *)(b4s + L + u_loc) = make_float4(e4[0], e4[1], e4[2], e4[3]);
                    *(float4 *)(b4s + L + u_loc + 4) = make_float4(e4[4], e4[5], e4[6], e4[7]);
                }
                __syncthreads();
                float b5[8];
                const float4 a = *(const float4 *)(b4s + u_loc + 16), c = *(const float4 *)(b4s + u_loc + 20);
                const float hi[8] = {a.x, a.y, a.z, a.w, c.x, c.y, c.z, c.w};
#pragma unroll
                for (int i = 0; i < 8; ++i) b5[i] = __fadd_rn(b4[i], hi[i]);
                GSP_SCAN_LEVEL(b5, 5)
            }
        }

        // ---- the block's winner: lanes, then warps (larger snr, then smaller (j, u) code)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float s = __shfl_xor_sync(0xffffffffu, best.snr, o);
            const int c = __shfl_xor_sync(0xffffffffu, best.code, o);
            if (better(s, c, best.snr, best.code)) {
                best.snr = s;
                best.code = c;
            }
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
        // (the next iteration's stage_block starts with loads and shuffles; its first shared-memory write that
        //  could clash — red[] — comes after every thread has passed the barrier above)
    }
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

__global__ void __launch_bounds__(256)
search_write_kernel(const float *__restrict__ best_snr, const int32_t *__restrict__ best_code, int64_t nblk, int L,
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
                c_dm[k] = d;
                c_u[k] = (int32_t)(b * L + (code & 0xffff));
                c_w[k] = 1 << (code >> 16);
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
                                                      s->d_best_snr, s->d_best_code, d_stats)
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
        search_write_kernel<<<s->ndm, 256, 0, st>>>(s->d_best_snr, s->d_best_code, s->nblk, s->L, s->threshold,
                                                    s->d_row_off, s->max_cand, d_cand_dm, d_cand_sample,
                                                    d_cand_width, d_cand_snr);
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
    cudaFree(s->d_row_count);
    cudaFree(s->d_row_off);
    cudaGetLastError();
    delete s;
    return GSP_OK;
}

}  // extern "C"
