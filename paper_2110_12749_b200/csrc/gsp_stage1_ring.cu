// gsp_stage1_ring.cu — streaming ("rolling window") stage-1 kernel for uint8 input.
//
//   S_s[t]  = sum_{c in subband s} x[t + s1[c]][c]      (Algorithm 1/2 of the paper applied per
//   S'_s[u] = sum_{k<ds} S_s[u*ds + k]   (un-divided)     subband: PAPER.md:104-166, sub-band
//                                                         method PAPER.md:100)
//
// Algorithm 1 of the paper walks the time axis with a lastdata/data pair so that every input
// sample is read once; this kernel is that idea on one SM.  A CTA owns 64 consecutive channels
// and a long time segment and keeps the last kRing = 1024 input rows of its channels in shared
// memory, TRANSPOSED to channel-major (ring position = input row mod 1024, the same for every
// channel).  Per chunk of 256 rows:
//
//   load      a lane reads 8 channels x 4 consecutive rows with four 64-bit loads (a warp request
//             covers 4 rows x one 64-byte segment), transposes two 4x4 byte blocks in registers
//             (16 PRMT) and stores eight words "one channel x 4 consecutive rows" into the ring;
//             the loads of the next chunk are issued before the current chunk is gathered.
//   gather    output t of channel c needs ring bytes (t + s1[c]) .. +3: lanes take consecutive
//             output words, read the two ring words that hold them (bank-conflict free for any
//             shift) and realign with PRMT.F4E; four samples per word are summed in two u16x2
//             accumulators (even / odd bytes).  A warp owns 16 channels x 32 output words.
//   reduce    the four 16-channel partial sums meet in shared memory, ds consecutive samples are
//             folded with shuffles and the result is written in the format stage 2 reads.
//
// Every input byte is fetched once (no halo re-reads between time tiles), the ring needs no
// per-channel window bookkeeping, and a group qualifies when its largest shift fits the ring
// (max s1 + 4 <= 768 rows); other groups run the windowed tile kernel of gsp_stage1.cu.

#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <cstdlib>

#include "gsp_internal.h"

namespace gsp {

namespace {

constexpr int kCG = 64;                 // channels per CTA
constexpr int kRing = 1024;             // ring length in rows (= bytes per channel)
constexpr int kRW = kRing / 4;          // ring words per channel
constexpr int kPitch = kRW + 1;         // word kRW mirrors word 0 (the realigning read of word 255)
constexpr int kChunk = 256;             // rows per chunk
constexpr int kChunkW = kChunk / 4;     // 64 quads / output words per chunk
constexpr int kThreadsR = 256;
constexpr int kRingWords = kCG * kPitch + 8;   // +4 words of skew for channels >= 32 (bank spread)
constexpr int kSmemRing = kRingWords * 4 + 4 * kChunkW * 8;   // ring + part[4][64] uint2

__device__ __forceinline__ uint32_t prmt_f4e(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("prmt.b32.f4e %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}


// 4x4 byte transpose: v[i] = row i (bytes = 4 channels) -> o[k] = channel k (bytes = 4 rows)
__device__ __forceinline__ void transpose4(uint32_t v0, uint32_t v1, uint32_t v2, uint32_t v3, uint32_t *o) {
    const uint32_t ta = __byte_perm(v0, v1, 0x5140), tb = __byte_perm(v0, v1, 0x7362);
    const uint32_t tc = __byte_perm(v2, v3, 0x5140), td = __byte_perm(v2, v3, 0x7362);
    o[0] = __byte_perm(ta, tc, 0x5410);
    o[1] = __byte_perm(ta, tc, 0x7632);
    o[2] = __byte_perm(tb, td, 0x5410);
    o[3] = __byte_perm(tb, td, 0x7632);
}

}  // namespace

namespace {

template <int FMT, int NCHAN>
__global__ void __launch_bounds__(kThreadsR, 3)
stage1_ring_u8_kernel(const uint8_t *__restrict__ x, const int32_t *__restrict__ s1, void *__restrict__ ws,
                      int64_t ws_pitch, int64_t n1d, int64_t nsamp, int nchan, int cps, int ds, int M,
                      const int2 *__restrict__ glist, int nglist, int64_t seg_rows) {
    extern __shared__ __align__(16) uint32_t smem_ring[];
    uint32_t *xs = smem_ring;                                  // [kCG][kPitch] (+ skew)
    uint2 *part = (uint2 *)(smem_ring + kRingWords);           // [4 slices][kChunkW]

    const int gi = blockIdx.x % nglist;
    const int64_t seg = blockIdx.x / nglist;
    const int2 ge = __ldg(glist + gi);
    const int group = ge.x, L = ge.y;                          // chunks resident before a gather
    const int cfirst = group * kCG;
    const int64_t total = n1d * ds;                            // S-samples that feed an output
    const int64_t ta = seg * seg_rows;                         // multiple of kRing
    if (ta >= total) return;
    const int64_t tb = (ta + seg_rows < total) ? ta + seg_rows : total;
    const int nk = (int)((tb - ta + kChunk - 1) / kChunk);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t nc = NCHAN ? NCHAN : nchan;

    // ---- load-side constants: lane = (8-channel column l8, row quad g)
    const int l8 = lane & 7, g = lane >> 3;
    const uint8_t *src = x + cfirst + 8 * l8;
    uint32_t *sdst = xs + (8 * l8) * kPitch + 4 * (l8 >> 2);
    const int Q0 = 8 * warp + g;                               // quads Q0 and Q0 + 4 of a chunk

    auto prefetch = [&](int jj, uint2 (&v)[2][4]) {
        const int64_t r0 = ta + (int64_t)kChunk * jj + 4 * Q0;
        const uint8_t *p = src + r0 * nc;
        if (ta + (int64_t)kChunk * (jj + 1) <= nsamp) {
#pragma unroll
            for (int q = 0; q < 2; ++q)
#pragma unroll
                for (int i = 0; i < 4; ++i) v[q][i] = __ldg((const uint2 *)(p + (16 * q + i) * nc));
        } else {
#pragma unroll
            for (int q = 0; q < 2; ++q)
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    v[q][i] = (r0 + 16 * q + i < nsamp) ? __ldg((const uint2 *)(p + (16 * q + i) * nc))
                                                        : make_uint2(0u, 0u);
        }
    };
    auto commit = [&](int jj, const uint2 (&v)[2][4]) {
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            uint32_t o[8];
            transpose4(v[q][0].x, v[q][1].x, v[q][2].x, v[q][3].x, o);
            transpose4(v[q][0].y, v[q][1].y, v[q][2].y, v[q][3].y, o + 4);
            const int pos = (kChunkW * jj + Q0 + 4 * q) & (kRW - 1);
            uint32_t *d = sdst + pos;
#pragma unroll
            for (int k = 0; k < 8; ++k) d[k * kPitch] = o[k];
            if (pos == 0) {
#pragma unroll
                for (int k = 0; k < 8; ++k) d[k * kPitch + kRW] = o[k];
            }
        }
    };

    // ---- gather-side constants: warp = (16-channel slice, 32-word half of the chunk)
    const int slice = warp & 3, half = warp >> 2;
    int sc[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) sc[j] = __ldg(s1 + cfirst + 16 * slice + j);
    const uint8_t *cb = (const uint8_t *)(xs + (16 * slice) * kPitch + 4 * (slice >> 1));
    const uint32_t lane_b = 128u * half + 4u * lane;

    // ---- reduce-side constants
    const int nsb = kCG / cps, sps = cps / 16;
    const uint16_t *part16 = (const uint16_t *)part;
    auto emit = [&](int s, int64_t u, int v) {
        if (u >= n1d) return;
        if (FMT == WS_I32) {
            ((int32_t *)ws)[(int64_t)s * ws_pitch + u] = v;
        } else {  // WS_PK16: W[i] = S'[i] | S'[i+M] << 16
            uint16_t *h = (uint16_t *)ws + 2 * ((int64_t)s * ws_pitch);
            h[2 * u] = (uint16_t)v;
            if (u >= M) h[2 * (u - M) + 1] = (uint16_t)v;
        }
    };

    uint2 v[2][4];
    for (int jj = 0; jj < L; ++jj) {
        prefetch(jj, v);
        commit(jj, v);
    }
    __syncthreads();

    for (int k = 0; k < nk; ++k) {
        prefetch(k + L, v);                                    // lands while chunk k is gathered

        // ------------------------------ gather chunk k ------------------------------
        const uint32_t Tb = (((uint32_t)k * kChunk) & (kRing - 1)) + lane_b;
        uint32_t E = 0u, O = 0u;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const uint32_t B = Tb + (uint32_t)sc[j];
            const uint32_t A = B & (kRing - 4);
            const uint8_t *p = cb + j * (kPitch * 4) + A;
            const uint32_t w = prmt_f4e(*(const uint32_t *)p, *(const uint32_t *)(p + 4), B);
            E += __byte_perm(w, 0u, 0x4240);                   // bytes 0 and 2 -> u16 lanes
            O += __byte_perm(w, 0u, 0x4341);                   // bytes 1 and 3 -> u16 lanes
        }
        part[slice * kChunkW + 32 * half + lane] =
            make_uint2(__byte_perm(E, O, 0x5410), __byte_perm(E, O, 0x7632));
        __syncthreads();                                       // chunk k's ring slot is free

        commit(k + L, v);

        // --------------------- slice reduce + downsample + store ---------------------
        {
            const int i = threadIdx.x;
            const int64_t t = ta + (int64_t)kChunk * k + i;
            for (int sb = 0; sb < nsb; ++sb) {
                int tot = 0;
                for (int sl = 0; sl < sps; ++sl) tot += (int)part16[(sb * sps + sl) * kChunk + i];
                for (int o = 1; o < ds; o <<= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
                if ((i & (ds - 1)) == 0) emit(group * nsb + sb, t / ds, tot);
            }
        }
        __syncthreads();                                       // ring stores visible, part[] free
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
static int env_int_ring(const char *name, int dflt) {
    const char *v = std::getenv(name);
    return v ? std::atoi(v) : dflt;
}

bool stage1_ring_supported(const gsp_plan &p) {
    if (p.dtype != GSP_U8) return false;
    if (p.nchan % kCG != 0) return false;
    if (!(p.cps == 16 || p.cps == 32 || p.cps == 64)) return false;
    const int d = p.ds;
    if (!(d == 1 || d == 2 || d == 4 || d == 8 || d == 16)) return false;
    return env_int_ring("GSP_S1_RING", 1) != 0;
}

// Split the 64-channel groups of a plan: groups whose largest stage-1 shift fits the ring go to
// the streaming kernel ({group, chunks resident before a gather}), the rest to the windowed one.
void plan_stage1_groups(gsp_plan &p) {
    p.g_ring.clear();
    p.g_win.clear();
    const int ngroups = (p.nchan + kCG - 1) / kCG;
    const bool ring = stage1_ring_supported(p);
    for (int g = 0; g < ngroups; ++g) {
        int mx = 0;
        for (int c = g * kCG; c < std::min(p.nchan, (g + 1) * kCG); ++c) mx = std::max(mx, p.s1[c]);
        if (ring && mx <= kRing - kChunk) {
            p.g_ring.push_back(make_int2(g, (mx + kChunk - 1) / kChunk + 1));
        } else {
            p.g_win.push_back(g);
        }
    }
    // time segments of the streaming kernel: about six waves of 3 CTAs per SM, each segment a
    // multiple of the ring length and long against its warm-up (<= 1024 rows)
    const int64_t total = p.n1d * (int64_t)p.ds;
    int64_t seg = env_int_ring("GSP_S1_SEG_ROWS", 0);
    if (seg <= 0) {
        const int64_t want = std::max<int64_t>(1, (int64_t)p.sm_count * 3 * 6 / std::max<size_t>(1, p.g_ring.size()));
        seg = (total + want - 1) / want;
        seg = std::max<int64_t>(seg, 8 * kRing);
    }
    seg = (seg + kRing - 1) / kRing * kRing;
    p.ring_seg_rows = seg;
    p.ring_nseg = std::max<int64_t>(1, (total + seg - 1) / seg);
}

typedef void (*Stage1RingFn)(const uint8_t *, const int32_t *, void *, int64_t, int64_t, int64_t, int, int,
                             int, int, const int2 *, int, int64_t);

template <int FMT>
static Stage1RingFn pick_ring_nchan(int nchan) {
    switch (nchan) {  // common filterbank widths get immediate row offsets
        case 4096: return stage1_ring_u8_kernel<FMT, 4096>;
        case 2048: return stage1_ring_u8_kernel<FMT, 2048>;
        case 1024: return stage1_ring_u8_kernel<FMT, 1024>;
        case 512: return stage1_ring_u8_kernel<FMT, 512>;
        default: return stage1_ring_u8_kernel<FMT, 0>;
    }
}

cudaError_t configure_stage1_ring(const gsp_plan &p) {
    if (p.g_ring.empty()) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute((const void *)pick_ring_nchan<WS_I32>(p.nchan),
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemRing);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute((const void *)pick_ring_nchan<WS_PK16>(p.nchan),
                                cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemRing);
}

cudaError_t launch_stage1_ring(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    if (p.g_ring.empty()) return cudaSuccess;
    Stage1RingFn fn = (p.ws_format == WS_PK16) ? pick_ring_nchan<WS_PK16>(p.nchan)
                    : (p.ws_format == WS_I32) ? pick_ring_nchan<WS_I32>(p.nchan) : nullptr;
    if (!fn) return cudaErrorInvalidValue;
    const int64_t nblocks = (int64_t)p.g_ring.size() * p.ring_nseg;
    if (nblocks > 0x7fffffff) return cudaErrorInvalidValue;
    fn<<<(unsigned)nblocks, kThreadsR, kSmemRing, st>>>((const uint8_t *)d_in, p.d_s1, p.d_ws, p.ws_pitch,
                                                        p.n1d, p.nsamp, p.nchan, p.cps, p.ds, p.t2.M,
                                                        p.d_g_ring, (int)p.g_ring.size(), p.ring_seg_rows);
    return cudaPeekAtLastError();
}

}  // namespace gsp
