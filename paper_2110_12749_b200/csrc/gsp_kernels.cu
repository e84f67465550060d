// gsp_kernels.cu — CUDA kernels (sm_100a) of the two dedispersion stages and their launchers.
//
//   stage 1  S_s[t]  = sum_{c in subband s} x[t + s1[c]][c]      (Alg. 1/2 per subband,
//   downsamp S'_s[u] = sum_{k<ds} S_s[u*ds + k]   (un-divided)     PAPER.md:104-166, :100)
//   stage 2  y_d[u]  = (1/ds) * sum_s S'_s[u + s2[d][s]]          (Alg. 2 with channels :=
//                                                                  subbands; float32 out :206)
//
// Two implementations per stage: "generic" = one thread per output with global loads
// (Algorithm 2 as printed, applied twice) and "tiled" = shared-memory staged kernels
// designed for B200.  uint8 input is summed in integers (exact); float32
// input in float32.

#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <type_traits>

#include "gsp_internal.h"
#include "gsp_device.cuh"

namespace gsp {

// y = fl32( tot / ds ) with the rounding of DESIGN.md §3: exact for ds a power of two;
// otherwise fl32( fl64(tot) * fl64(1/ds) ).
struct OutScale {
    int mode;     // 0: ds == 1, 1: power of two, 2: general
    float f;      // 1/ds as float (modes 1, and float32 input)
    double d;     // 1/ds as double (mode 2)
};

__device__ __forceinline__ float scale_int(int v, const OutScale &sc) {
    if (sc.mode == 0) return (float)v;
    if (sc.mode == 1) return (float)v * sc.f;
    return (float)((double)v * sc.d);
}

// ====================================================================================
// generic stage 1 (+ downsample epilogue): one thread per S'_s[u]
// ====================================================================================
// RFI: the prologue F1/F4 of gsp_rfi.cu applied at the loads (uint8 only): masked channels and clipped rows
// read as the channel's pad value.
struct RfiArgs {
    const uint32_t *clip_bits;
    const uint8_t *chan_mask, *chan_pad;
};

template <typename TIn, int FMT, bool RFI>
__global__ void __launch_bounds__(256)
stage1_generic_kernel(const TIn *__restrict__ x, const int32_t *__restrict__ s1, void *__restrict__ ws,
                      int64_t ws_pitch, int64_t n1d, int nchan, int cps, int ds, int M, RfiArgs rfi,
                      const int32_t *__restrict__ sub_list) {
    extern __shared__ int32_t sh_s1[];
    const int s = sub_list ? sub_list[blockIdx.y] : (int)blockIdx.y;
    for (int j = threadIdx.x; j < cps; j += blockDim.x) sh_s1[j] = s1[s * cps + j];
    __syncthreads();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= n1d) return;
    typedef typename std::conditional<std::is_same<TIn, float>::value, float, int>::type Acc;
    Acc tot = 0;
    for (int k = 0; k < ds; ++k) {
        const int64_t t = u * ds + k;
        const TIn *col = x + (int64_t)s * cps;
        if (RFI) {
            for (int j = 0; j < cps; ++j) {
                const int64_t r = t + sh_s1[j];
                const int c = s * cps + j;
                const bool sub = (rfi.chan_mask && rfi.chan_mask[c]) ||
                                 (rfi.clip_bits && ((rfi.clip_bits[r >> 5] >> (unsigned)(r & 31)) & 1u));
                tot += sub ? (Acc)rfi.chan_pad[c] : (Acc)col[r * (int64_t)nchan + j];
            }
        } else {
            for (int j = 0; j < cps; ++j) tot += (Acc)col[(t + sh_s1[j]) * (int64_t)nchan + j];
        }
    }
    if (FMT == WS_I32) {
        ((int32_t *)ws)[(int64_t)s * ws_pitch + u] = (int32_t)tot;
    } else if (FMT == WS_F32) {
        ((float *)ws)[(int64_t)s * ws_pitch + u] = (float)tot;
    } else {  // WS_PK16: W[i] = S'[i] | S'[i+M] << 16, little-endian halves
        uint16_t *h = (uint16_t *)ws + 2 * ((int64_t)s * ws_pitch);
        h[2 * u] = (uint16_t)tot;
        if (u >= M) h[2 * (u - M) + 1] = (uint16_t)tot;
    }
}

// ====================================================================================
// generic stage 2 (+ store epilogue): one thread per y_d[u]
// ====================================================================================
template <int FMT>
__global__ void __launch_bounds__(256)
stage2_generic_kernel(const void *__restrict__ ws, int64_t ws_pitch, const int32_t *__restrict__ s2,
                      float *__restrict__ out, int64_t out_pitch, int64_t nout, int nsub, OutScale sc) {
    extern __shared__ int32_t sh_s2[];
    const int d = blockIdx.y;
    for (int s = threadIdx.x; s < nsub; s += blockDim.x) sh_s2[s] = s2[(int64_t)d * nsub + s];
    __syncthreads();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= nout) return;
    float *dst = out + (int64_t)d * out_pitch + u;
    if (FMT == WS_F32) {
        const float *w = (const float *)ws;
        float tot = 0.f;
        for (int s = 0; s < nsub; ++s) tot += w[(int64_t)s * ws_pitch + u + sh_s2[s]];
        *dst = tot * sc.f;
    } else if (FMT == WS_I32) {
        const int32_t *w = (const int32_t *)ws;
        int tot = 0;
        for (int s = 0; s < nsub; ++s) tot += w[(int64_t)s * ws_pitch + u + sh_s2[s]];
        *dst = scale_int(tot, sc);
    } else {
        const uint32_t *w = (const uint32_t *)ws;
        int tot = 0;
        for (int s = 0; s < nsub; ++s) tot += (int)(w[(int64_t)s * ws_pitch + u + sh_s2[s]] & 0xffffu);
        *dst = scale_int(tot, sc);
    }
}

// ====================================================================================
// tiled stage 2 (uint8 path): persistent, warp-specialised, bulk-copy fed
// ====================================================================================
// One CTA tile = Q trial DMs x T = 2*M output samples.  The subband intermediate is
// stored "planar-packed": word i of subband s holds S'_s[i] in its low half and
// S'_s[i+M] in its high half, so the operand of output pair (u0+w, u0+M+w) for ANY
// shift is the single 32-bit word W_s[u0 + w + shift] — every shift is word aligned and
// one 32-bit integer add performs two subband adds.  Lanes take consecutive words
// (bank-conflict free for every shift).  Four subbands are summed in 16-bit lanes
// (4 * cps*255*ds <= 65535), then folded into 32-bit accumulators:
//     all += p            (mod 2^32: lo_sum + 65536*hi_sum)
//     hi  += p >> 16
// and lo_sum = all - (hi << 16) at the end.  A producer warp streams the windows of the next
// subband chunks with cp.async.bulk (TMA engine, SASS UBLKCP) through an nstage ring guarded
// by full/empty mbarriers; the ring runs across tile boundaries so it never drains.  The
// consumers never wait on a round trip between chunks: the release is a fire-and-forget
// arrive and the next stage's barrier is polled while the current chunk's loads are in
// flight (measured: every synchronous hop through the saturated load/store queue costs
// ~650 cycles).  setmaxnreg moves registers from the producer warpgroup to the consumers.
constexpr int kConsumerWarps = 16;
constexpr int kProducerWarps = 4;  // one warpgroup: warp 0 issues the copies, warps 1-3 retire at once
constexpr int kStage2Threads = (kConsumerWarps + kProducerWarps) * 32;
constexpr int kMaxStages = 8;
constexpr int kConsumerRegs = 112;  // setmaxnreg only redistributes the registers the CTA was launched with:
                                    // 5 warpgroups * 96 = 480 >= 4 * 112 + 24
constexpr int kProducerRegs = 24;

template <int DPW, int WPL, int MODE>
__global__ void __launch_bounds__(kStage2Threads, 1)
stage2_tiled_kernel(const uint32_t *__restrict__ W, int64_t ws_pitch, const int4 *__restrict__ prod,
                    const int32_t *__restrict__ offs, const int32_t *__restrict__ rows,
                    float *__restrict__ out, int64_t out_pitch, int64_t nout, int nsub, int nchunk,
                    int ndmblk, int64_t ntiles, int nstage, int stage_words, OutScale sc) {
    constexpr bool F32 = (MODE == S2_F32);
    constexpr bool PACKED = (MODE <= S2_PK1);
    constexpr int Q = kConsumerWarps * DPW;
    constexpr int M = 32 * WPL;
    constexpr int TT = PACKED ? 2 * M : M;   // outputs per tile: packed words hold two samples, int32 / float32 words one
    extern __shared__ __align__(128) uint8_t smem_raw[];
    uint64_t *full = (uint64_t *)smem_raw;   // [kMaxStages] copy landed (tx bytes)
    uint64_t *empty = full + kMaxStages;     // [kMaxStages] all consumer warps released the stage
    uint32_t *buf = (uint32_t *)(smem_raw + 256);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int i = 0; i < nstage; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], kConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp < kProducerWarps) {
        // ------------------------------ producer warpgroup ------------------------------
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kProducerRegs));
        if (warp != 0) return;
        int st = 0;
        uint32_t ph = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const int64_t tt = tile / ndmblk;
            const int blk = (int)(tile - tt * ndmblk);
            const int64_t u0 = tt * TT;
            for (int ch = 0; ch < nchunk; ++ch) {
                const int s = ch * 4 + (lane & 3);
                const int4 pr = __ldg(prod + (int64_t)blk * nsub + s);   // {start, words, offset}
                const uint32_t bytes = (uint32_t)pr.y * 4u;
                uint32_t total = bytes + __shfl_xor_sync(0xffffffffu, bytes, 1);
                total += __shfl_xor_sync(0xffffffffu, total, 2);
                mbar_wait(&empty[st], ph ^ 1u);
                if (lane == 0) mbar_arrive_expect_tx(&full[st], total);
                __syncwarp();
                if (lane < 4)
                    bulk_g2s(buf + (size_t)st * stage_words + pr.z,
                             W + (int64_t)s * ws_pitch + u0 + pr.x, bytes, &full[st]);
                if (++st == nstage) {
                    st = 0;
                    ph ^= 1u;
                }
            }
        }
        return;
    }

    // --------------------------------- consumer warps ---------------------------------
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kConsumerRegs));
    const int cw = warp - kProducerWarps;
    int st = 0;
    uint32_t ph = 0;
    bool ready = false;   // full[st] already seen complete (tested during the previous chunk)
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t tt = tile / ndmblk;
        const int blk = (int)(tile - tt * ndmblk);
        const int64_t u0 = tt * TT;
        const int dq0 = blk * Q + cw * DPW;

        // packed path: acc_all / acc_hi as described above; int32 / float32 paths: acc_all holds the sums
        uint32_t acc_all[DPW][WPL], acc_hi[PACKED ? DPW : 1][PACKED ? WPL : 1];
#pragma unroll
        for (int dd = 0; dd < DPW; ++dd)
#pragma unroll
            for (int j = 0; j < WPL; ++j) {
                acc_all[dd][j] = 0u;
                if (PACKED) acc_hi[dd][j] = 0u;
            }

        int4 o_next[DPW];
#pragma unroll
        for (int dd = 0; dd < DPW; ++dd)
            o_next[dd] = __ldg((const int4 *)(offs + (int64_t)(dq0 + dd) * nsub));

        for (int ch = 0; ch < nchunk; ++ch) {
            int4 o[DPW];
#pragma unroll
            for (int dd = 0; dd < DPW; ++dd) o[dd] = o_next[dd];
            if (ch + 1 < nchunk) {
#pragma unroll
                for (int dd = 0; dd < DPW; ++dd)
                    o_next[dd] = __ldg((const int4 *)(offs + (int64_t)(dq0 + dd) * nsub + (ch + 1) * 4));
            }
            if (!ready) mbar_wait(&full[st], ph);
            // Poll the NEXT stage's barrier now: its round trip through the load/store queue
            // overlaps this chunk's loads instead of stalling the warp between chunks.
            const int st_n = (st + 1 == nstage) ? 0 : st + 1;
            const uint32_t ph_n = (st + 1 == nstage) ? (ph ^ 1u) : ph;
            ready = mbar_test_wait(&full[st_n], ph_n);

            const uint32_t *sb = buf + (size_t)st * stage_words + lane;
#pragma unroll
            for (int dd = 0; dd < DPW; ++dd) {
                const uint32_t *b0 = sb + o[dd].x;
                const uint32_t *b1 = sb + o[dd].y;
                const uint32_t *b2 = sb + o[dd].z;
                const uint32_t *b3 = sb + o[dd].w;
#pragma unroll
                for (int j = 0; j < WPL; ++j) {
                    if (F32) {
                        const float p = (__uint_as_float(b0[32 * j]) + __uint_as_float(b1[32 * j])) +
                                        (__uint_as_float(b2[32 * j]) + __uint_as_float(b3[32 * j]));
                        acc_all[dd][j] = __float_as_uint(__uint_as_float(acc_all[dd][j]) + p);
                    } else if (MODE == S2_I32) {
                        acc_all[dd][j] += (b0[32 * j] + b1[32 * j]) + (b2[32 * j] + b3[32 * j]);
                    } else if (MODE == S2_PK4) {
                        const uint32_t p = (b0[32 * j] + b1[32 * j]) + (b2[32 * j] + b3[32 * j]);
                        acc_all[dd][j] += p;
                        acc_hi[dd][j] += p >> 16;
                    } else if (MODE == S2_PK2) {   // a 16-bit lane holds two subband sums at most
                        const uint32_t p = b0[32 * j] + b1[32 * j], q = b2[32 * j] + b3[32 * j];
                        acc_all[dd][j] += p + q;
                        acc_hi[dd][j] += (p >> 16) + (q >> 16);
                    } else {                       // S2_PK1: every subband sum is folded on its own
                        const uint32_t w0 = b0[32 * j], w1 = b1[32 * j], w2 = b2[32 * j], w3 = b3[32 * j];
                        acc_all[dd][j] += (w0 + w1) + (w2 + w3);
                        acc_hi[dd][j] += ((w0 >> 16) + (w1 >> 16)) + ((w2 >> 16) + (w3 >> 16));
                    }
                }
            }
            // release the stage: one fire-and-forget arrive per warp
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
            st = st_n;
            ph = ph_n;
        }

        // ------------------------------ store epilogue ------------------------------
#pragma unroll
        for (int dd = 0; dd < DPW; ++dd) {
            const int row = __ldg(rows + dq0 + dd);
            if (row < 0) continue;
            float *orow = out + (int64_t)row * out_pitch;
#pragma unroll
            for (int j = 0; j < WPL; ++j) {
                const int64_t u = u0 + lane + 32 * j;
                if (F32) {
                    if (u < nout) orow[u] = __uint_as_float(acc_all[dd][j]) * sc.f;
                } else if (MODE == S2_I32) {
                    if (u < nout) orow[u] = scale_int((int)acc_all[dd][j], sc);
                } else {
                    const uint32_t hi = acc_hi[dd][j];
                    const uint32_t lo = acc_all[dd][j] - (hi << 16);
                    if (u < nout) orow[u] = scale_int((int)lo, sc);
                    if (u + M < nout) orow[u + M] = scale_int((int)hi, sc);
                }
            }
        }
    }
}

// ====================================================================================
// launchers
// ====================================================================================
static OutScale make_scale(int ds) {
    OutScale sc;
    sc.f = 1.0f / (float)ds;
    sc.d = 1.0 / (double)ds;
    sc.mode = (ds == 1) ? 0 : (((ds & (ds - 1)) == 0) ? 1 : 2);
    return sc;
}

cudaError_t launch_stage1_generic(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    return launch_stage1_generic_list(p, d_in, nullptr, p.nsub, st);
}

cudaError_t launch_stage1_generic_list(const gsp_plan &p, const void *d_in, const int32_t *d_list, int nlist,
                                       cudaStream_t st) {
    if (nlist <= 0) return cudaSuccess;
    dim3 grid((unsigned)((p.n1d + 255) / 256), (unsigned)nlist);
    const size_t sh = (size_t)p.cps * sizeof(int32_t);
    const int M = p.t2.M;
    RfiArgs rfi = {p.rfi.d_clip_bits, p.rfi.d_mask, p.rfi.d_pad};
#define GSP_S1G(TIN, FMT, RFI)                                                                            \
    stage1_generic_kernel<TIN, FMT, RFI><<<grid, 256, sh, st>>>((const TIN *)d_in, p.d_s1, p.d_ws,        \
                                                                p.ws_pitch, p.n1d, p.nchan, p.cps, p.ds, \
                                                                M, rfi, d_list)
    if (p.dtype == GSP_F32) {
        GSP_S1G(float, WS_F32, false);
    } else if (p.rfi.enabled) {
        if (p.ws_format == WS_PK16) GSP_S1G(uint8_t, WS_PK16, true);
        else GSP_S1G(uint8_t, WS_I32, true);
    } else if (p.ws_format == WS_PK16) {
        GSP_S1G(uint8_t, WS_PK16, false);
    } else {
        GSP_S1G(uint8_t, WS_I32, false);
    }
#undef GSP_S1G
    return cudaPeekAtLastError();
}

cudaError_t launch_stage2_generic(const gsp_plan &p, float *d_out, cudaStream_t st) {
    dim3 grid((unsigned)((p.nout + 255) / 256), (unsigned)p.ndm);
    const size_t sh = (size_t)p.nsub * sizeof(int32_t);
    const OutScale sc = make_scale(p.ds);
#define GSP_S2G(FMT)                                                                           \
    stage2_generic_kernel<FMT><<<grid, 256, sh, st>>>(p.d_ws, p.ws_pitch, p.d_s2, d_out,       \
                                                      p.out_pitch, p.nout, p.nsub, sc)
    if (p.ws_format == WS_F32) {
        GSP_S2G(WS_F32);
    } else if (p.ws_format == WS_I32) {
        GSP_S2G(WS_I32);
    } else {
        GSP_S2G(WS_PK16);
    }
#undef GSP_S2G
    return cudaPeekAtLastError();
}

typedef void (*Stage2TiledFn)(const uint32_t *, int64_t, const int4 *, const int32_t *, const int32_t *,
                              float *, int64_t, int64_t, int, int, int, int64_t, int, int, OutScale);

template <int MODE>
static Stage2TiledFn pick_stage2_shape(int dpw, int wpl) {
    if (MODE >= S2_I32) {   // one operand per word
        if (dpw == 4 && wpl == 16) return stage2_tiled_kernel<4, 16, MODE>;
        if (dpw == 2 && wpl == 32) return stage2_tiled_kernel<2, 32, MODE>;
        if (dpw == 2 && wpl == 16) return stage2_tiled_kernel<2, 16, MODE>;
        if (dpw == 4 && wpl == 8) return stage2_tiled_kernel<4, 8, MODE>;
        if (dpw == 2 && wpl == 8) return stage2_tiled_kernel<2, 8, MODE>;
        if (dpw == 1 && wpl == 8) return stage2_tiled_kernel<1, 8, MODE>;
        if (dpw == 1 && wpl == 32) return stage2_tiled_kernel<1, 32, MODE>;
        if (dpw == 1 && wpl == 16) return stage2_tiled_kernel<1, 16, MODE>;
        return nullptr;
    }
    if (dpw == 2 && wpl == 16) return stage2_tiled_kernel<2, 16, MODE>;
    if (dpw == 1 && wpl == 32) return stage2_tiled_kernel<1, 32, MODE>;
    if (dpw == 4 && wpl == 8) return stage2_tiled_kernel<4, 8, MODE>;
    if (dpw == 1 && wpl == 16) return stage2_tiled_kernel<1, 16, MODE>;
    if (dpw == 2 && wpl == 8) return stage2_tiled_kernel<2, 8, MODE>;
    if (dpw == 1 && wpl == 8) return stage2_tiled_kernel<1, 8, MODE>;
    return nullptr;
}

static Stage2TiledFn pick_stage2_tiled(int Q, int M, int mode) {
    const int dpw = Q / kConsumerWarps, wpl = M / 32;
    switch (mode) {
        case S2_PK4: return pick_stage2_shape<S2_PK4>(dpw, wpl);
        case S2_PK2: return pick_stage2_shape<S2_PK2>(dpw, wpl);
        case S2_PK1: return pick_stage2_shape<S2_PK1>(dpw, wpl);
        case S2_I32: return pick_stage2_shape<S2_I32>(dpw, wpl);
        case S2_F32: return pick_stage2_shape<S2_F32>(dpw, wpl);
    }
    return nullptr;
}

// The dynamic shared-memory limit of a kernel is a per-function (process-wide) attribute: it is set to the
// device's opt-in maximum, never to one plan's need, so plans created in any order can share an instantiation.
cudaError_t configure_kernels(const gsp_plan &p) {
    if (!p.t2.supported) return cudaSuccess;
    Stage2TiledFn fn = pick_stage2_tiled(p.t2.Q, p.t2.M, p.t2.mode);
    if (!fn) return cudaErrorInvalidValue;
    return cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)p.smem_optin);
}

cudaError_t launch_stage2_tiled(const gsp_plan &p, float *d_out, cudaStream_t st) {
    const Stage2Tiling &t = p.t2;
    Stage2TiledFn fn = pick_stage2_tiled(t.Q, t.M, t.mode);
    if (!fn) return cudaErrorInvalidValue;
    const int64_t ntiles = t.ntile_t * (int64_t)t.ndmblk;
    const unsigned grid = (unsigned)std::min<int64_t>(ntiles, (int64_t)p.sm_count);
    fn<<<grid, kStage2Threads, t.smem_bytes, st>>>((const uint32_t *)p.d_ws, p.ws_pitch, p.d_t2_prod,
                                                   p.d_t2_offs, p.d_t2_rows, d_out, p.out_pitch,
                                                   p.nout, p.nsub, t.nchunk, t.ndmblk, ntiles,
                                                   t.nstage, t.stage_words, make_scale(p.ds));
    return cudaPeekAtLastError();
}

}  // namespace gsp
