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
#include "gsp_device.cuh"

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
// TMA-fed variant of the streaming kernel (the one gsp_dedisperse runs).
//
// Same ring, gather and reduce as above; what changes is how the input reaches the ring.  A
// producer warp streams 128-row x 64-byte boxes of the time-major input into a kNStage-deep
// shared-memory ring with 2-D tiled TMA loads (cp.async.bulk.tensor, SASS UTMALDG), guarded by
// full/empty mbarriers, so kNStage*8 KB per CTA are in flight whatever the eight consumer warps
// are doing.  The byte transposition is done by the load itself: ldmatrix.m16n16.trans.b8 (new on
// sm_100) hands thread t of a warp the two words "channel t/4 (+8), rows 4(t%4)..+3" of a 16-row x
// 16-channel tile of the landed stage, i.e. ring words, which the lanes store channel-major into
// the ring (pitch = 4 mod 32: the 8 channels x 4 quads of a fragment hit 32 banks).  The boxes are
// written with the TMA 64-byte swizzle so that the sixteen 16-byte rows an ldmatrix reads (64 bytes
// apart) fall on all eight 16-byte bank groups.  Rows past the end of the input are zero-filled by
// the TMA unit (they only ever feed S-samples that are not emitted).
// ---------------------------------------------------------------------------------------------
namespace {

constexpr int kHalf = 128;                       // rows per TMA stage (half a chunk)
constexpr int kStageBytes = kHalf * kCG;         // 8 KB
constexpr int kNStage = 5;
constexpr int kConsumerThreads = 256;            // 8 warps; warp 8 is the producer
constexpr int kThreadsT = kConsumerThreads + 32;
constexpr int kPitchL = kRW + 4;                 // ring pitch of this kernel: = 4 mod 32, so the 32 lanes of an ldmatrix
                                                 // fragment store (8 channels x 4 quads) hit 32 banks
constexpr int kRingWordsL = kCG * kPitchL;
// barriers | (up to 1 KB of alignment slack) | stages, 1 KB aligned for the TMA swizzle | ring | part
constexpr int kSmemStream = 128 + 1024 + kNStage * kStageBytes + kRingWordsL * 4 + 4 * kChunkW * 8;

template <int FMT, int CPS>
__global__ void __launch_bounds__(kThreadsT, 2)
stage1_stream_u8_kernel(const __grid_constant__ CUtensorMap tmap, const int32_t *__restrict__ s1,
                        void *__restrict__ ws, int64_t ws_pitch, int64_t n1d, int cps_unused, int ds, int lds, int M,
                        const int2 *__restrict__ glist, int nglist, int64_t seg_rows) {
    extern __shared__ __align__(128) uint8_t smem_stream[];
    uint64_t *full = (uint64_t *)smem_stream;                  // [kNStage] box landed (tx bytes)
    uint64_t *empty = full + 8;                                // [kNStage] all consumer warps have read it
    // stages: [kNStage][kHalf rows][64 B] time-major, written by TMA with the 64-byte swizzle (16-byte chunk
    // index ^= (row >> 1) & 3), which needs the buffer on a 1 KB boundary of the shared address space
    uint8_t *stage = smem_stream + 128 + ((1024u - ((smem_u32(smem_stream) + 128u) & 1023u)) & 1023u);
    uint32_t *xs = (uint32_t *)(stage + kNStage * kStageBytes);   // [kCG][kPitchL] channel-major ring
    uint2 *part = (uint2 *)(xs + kRingWordsL);                 // [4 slices][kChunkW]

    const int gi = blockIdx.x % nglist;
    const int64_t seg = blockIdx.x / nglist;
    const int2 ge = __ldg(glist + gi);
    const int group = ge.x, L = ge.y;                          // chunks resident before a gather
    const int cfirst = group * kCG;
    const int64_t total = n1d << lds;                          // S-samples that feed an output
    const int64_t ta = seg * seg_rows;                         // multiple of kRing
    if (ta >= total) return;
    const int64_t tb = (ta + seg_rows < total) ? ta + seg_rows : total;
    const int nk = (int)((tb - ta + kChunk - 1) / kChunk);
    const int nhalf = 2 * (nk + L);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int i = 0; i < kNStage; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], kConsumerThreads / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == kConsumerThreads / 32) {
        // ------------------------------------ producer ------------------------------------
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            for (int h = 0; h < nhalf; ++h) {
                while (!mbar_try_wait(&empty[st], ph ^ 1u)) __nanosleep(64);   // do not steal issue slots
                mbar_arrive_expect_tx(&full[st], kStageBytes);
                tma_load_2d(stage + st * kStageBytes, &tmap, cfirst, (int)(ta + (int64_t)kHalf * h), &full[st]);
                if (++st == kNStage) {
                    st = 0;
                    ph ^= 1u;
                }
            }
        }
        return;
    }

    // ---- commit: ldmatrix.trans on bytes.  A warp owns 16 rows of the landed stage (row block = warp) and walks
    //      the four 16-channel blocks; one ldmatrix.m16n16.trans.b8 hands thread t the ring words
    //      "channel t/4, rows 4(t%4)..+3" and "channel t/4 + 8, same rows" of the 16 x 16 byte tile: the byte
    //      transposition costs no ALU instruction at all.
    const int lrow = 16 * warp + (lane & 15);                  // the stage row this lane addresses for ldmatrix
    const uint32_t lsw = (uint32_t)((lrow >> 1) & 3);          // its swizzle term
    const uint32_t ld_off = (uint32_t)(lrow * kCG);
    const int qq = 4 * warp + (lane & 3);                      // quad of a half chunk (32 quads) this lane stores
    uint32_t *sdst = xs + (lane >> 2) * kPitchL;
    int cst = 0;
    uint32_t cph = 0;

    auto commit = [&](int h) {
        mbar_wait(&full[cst], cph);
        const uint32_t sbase = smem_u32(stage) + (uint32_t)(cst * kStageBytes) + ld_off;
        uint32_t o[8];
        // .x2: lanes 0-15 address the rows of channel block 2i, lanes 16-31 those of block 2i + 1
#pragma unroll
        for (int i = 0; i < 2; ++i)
            asm volatile("ldmatrix.sync.aligned.m16n16.x2.trans.shared.b8 {%0, %1, %2, %3}, [%4];"
                         : "=r"(o[4 * i]), "=r"(o[4 * i + 1]), "=r"(o[4 * i + 2]), "=r"(o[4 * i + 3])
                         : "r"(sbase + ((((uint32_t)(2 * i) + (uint32_t)(lane >> 4)) ^ lsw) << 4))
                         : "memory");
        // the stage is free once every lane's loads have returned
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[cst]);
        if (++cst == kNStage) {
            cst = 0;
            cph ^= 1u;
        }
        const int pos = (32 * h + qq) & (kRW - 1);
        uint32_t *d = sdst + pos;
#pragma unroll
        for (int cb = 0; cb < 4; ++cb) {
            d[(16 * cb) * kPitchL] = o[2 * cb];
            d[(16 * cb + 8) * kPitchL] = o[2 * cb + 1];
        }
        if (warp == 0 && (h & 7) == 0) {                       // warp-uniform: the quad that holds word 0
            if ((lane & 3) == 0) {
#pragma unroll
                for (int cb = 0; cb < 4; ++cb) {
                    d[(16 * cb) * kPitchL + kRW] = o[2 * cb];
                    d[(16 * cb + 8) * kPitchL + kRW] = o[2 * cb + 1];
                }
            }
        }
    };

    // ---- gather-side constants: warp = (16-channel slice, 32-word half of the chunk)
    const int slice = warp & 3, half = warp >> 2;
    int sc[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) sc[j] = __ldg(s1 + cfirst + 16 * slice + j);
    const uint8_t *cb = (const uint8_t *)(xs + (16 * slice) * kPitchL);
    const uint32_t lane_b = 128u * half + 4u * lane;

    // ---- reduce-side constants
    constexpr int nsb = kCG / CPS, sps = CPS / 16;     // subbands per group, 16-channel slices per subband
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

    for (int h = 0; h < 2 * L; ++h) commit(h);
    named_bar_sync(1, kConsumerThreads);

    for (int k = 0; k < nk; ++k) {
        // ------------------------------ gather chunk k ------------------------------
        const uint32_t Tb = (((uint32_t)k * kChunk) & (kRing - 1)) + lane_b;
        // T = sum of the words mod 2^32 = E + 256*O with E / O the u16x2 sums of the even / odd
        // bytes; E < 2^32, so E = T - (O << 8) exactly and only the odd bytes need unpacking.
        uint32_t Tq[4] = {0u, 0u, 0u, 0u}, Oq[4] = {0u, 0u, 0u, 0u};   // four independent add chains
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const uint32_t B = Tb + (uint32_t)sc[j];
            const uint32_t A = B & (kRing - 4);
            const uint8_t *p = cb + j * (kPitchL * 4) + A;
            const uint32_t w = prmt_f4e(*(const uint32_t *)p, *(const uint32_t *)(p + 4), B);
            Tq[j & 3] += w;
            Oq[j & 3] += __byte_perm(w, 0u, 0x4341);           // bytes 1 and 3 -> u16 lanes
        }
        const uint32_t T = (Tq[0] + Tq[1]) + (Tq[2] + Tq[3]);
        const uint32_t O = (Oq[0] + Oq[1]) + (Oq[2] + Oq[3]);
        const uint32_t E = T - (O << 8);
        part[slice * kChunkW + 32 * half + lane] =
            make_uint2(__byte_perm(E, O, 0x5410), __byte_perm(E, O, 0x7632));
        named_bar_sync(1, kConsumerThreads);                   // chunk k's ring slot is free

        commit(2 * (k + L));
        commit(2 * (k + L) + 1);

        // --------------------- slice reduce + downsample + store ---------------------
        {
            const int i = threadIdx.x;
            const int64_t t = ta + (int64_t)kChunk * k + i;
#pragma unroll
            for (int sb = 0; sb < nsb; ++sb) {
                int tot = 0;
#pragma unroll
                for (int sl = 0; sl < sps; ++sl) tot += (int)part16[(sb * sps + sl) * kChunk + i];
                for (int o = 1; o < ds; o <<= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
                if ((i & (ds - 1)) == 0) emit(group * nsb + sb, t >> lds, tot);
            }
        }
        named_bar_sync(1, kConsumerThreads);                   // ring stores visible, part[] free
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
    p.s_wide[0].clear();
    p.s_wide[1].clear();
    p.ns_wide[0] = p.ns_wide[1] = 0;
    const int ngroups = (p.nchan + kCG - 1) / kCG;
    const bool ring = stage1_ring_supported(p);
    const bool wide = stage1_wide_supported(p);
    for (int g = 0; g < ngroups; ++g) {
        int mx = 0;
        for (int c = g * kCG; c < std::min(p.nchan, (g + 1) * kCG); ++c) mx = std::max(mx, p.s1[c]);
        if (ring && mx <= kRing - kChunk) {
            p.g_ring.push_back(make_int2(g, (mx + kChunk - 1) / kChunk + 1));
            continue;
        }
        // shifts too large for the channel-major ring: the group's subbands stream through the wide
        // kernel when every one of them fits its time-major ring, else the windowed tile kernel
        const int s0 = g * kCG / p.cps, s1e = std::min(p.nsub, (g + 1) * kCG / p.cps);
        bool fits = wide && (g + 1) * kCG <= p.nchan;
        for (int s = s0; s < s1e && fits; ++s) fits = stage1_wide_slots(p, s) > 0;
        if (fits) {   // experiment switch: only groups at least this wide (in ring slots) leave the windowed kernel
            int mxs = 0;
            for (int s = s0; s < s1e; ++s) mxs = std::max(mxs, stage1_wide_slots(p, s));
            if (mxs < env_int_ring("GSP_S1_WIDE_MIN_SLOTS", 0)) fits = false;
        }
        if (!fits) {
            p.g_win.push_back(g);
            continue;
        }
        for (int s = s0; s < s1e; ++s) {
            const int ns = stage1_wide_slots(p, s);
            const int l = ns <= stage1_wide_mid_slots() ? 0 : 1;
            p.s_wide[l].push_back(s);
            p.ns_wide[l] = std::max(p.ns_wide[l], ns);
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

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)sym;
        cudaGetLastError();
    }
    return fn;
}

static bool stream_enabled() { return env_int_ring("GSP_S1_TMA", 1) != 0 && encode_tiled_fn() != nullptr; }

typedef void (*Stage1StreamFn)(const CUtensorMap, const int32_t *, void *, int64_t, int64_t, int, int, int, int,
                               const int2 *, int, int64_t);

template <int FMT>
static Stage1StreamFn pick_stream(int cps) {   // channels per subband are a template parameter of the reduce step
    switch (cps) {
        case 64: return (Stage1StreamFn)stage1_stream_u8_kernel<FMT, 64>;
        case 32: return (Stage1StreamFn)stage1_stream_u8_kernel<FMT, 32>;
        case 16: return (Stage1StreamFn)stage1_stream_u8_kernel<FMT, 16>;
        default: return nullptr;
    }
}

template <int FMT>
static cudaError_t set_stream_attr() {
    cudaError_t e = cudaSuccess;
    for (int cps = 16; cps <= 64 && e == cudaSuccess; cps *= 2)
        e = cudaFuncSetAttribute((const void *)pick_stream<FMT>(cps), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 kSmemStream);
    return e;
}

cudaError_t configure_stage1_ring(const gsp_plan &p) {
    if (p.g_ring.empty()) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute((const void *)pick_ring_nchan<WS_I32>(p.nchan),
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemRing);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute((const void *)pick_ring_nchan<WS_PK16>(p.nchan),
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemRing);
    if (e == cudaSuccess)
        e = set_stream_attr<WS_I32>();
    if (e == cudaSuccess)
        e = set_stream_attr<WS_PK16>();
    return e;
}

// The input as a 2-D tensor {nchan (innermost), nsamp}, fetched in boxes of box_chan channels x box_rows rows.
cudaError_t make_input_map(const gsp_plan &p, const void *d_in, int box_chan, int box_rows, CUtensorMap *tm,
                           bool swizzle64) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return cudaErrorNotSupported;
    const bool f32 = (p.dtype == GSP_F32);
    const cuuint64_t dims[2] = {(cuuint64_t)p.nchan, (cuuint64_t)p.nsamp};
    const cuuint64_t strides[1] = {(cuuint64_t)p.nchan * (f32 ? 4u : 1u)};
    const cuuint32_t box[2] = {(cuuint32_t)box_chan, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1u, 1u};
    static const CUtensorMapL2promotion promo[4] = {CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_64B,
                                                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B};
    const int pi = std::min(3, std::max(0, env_int_ring("GSP_TMA_L2_PROMOTION", 3)));
    const CUresult r = enc(tm, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_UINT8, 2,
                           const_cast<void *>(d_in), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           swizzle64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE, promo[pi],
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

bool tma_available() { return encode_tiled_fn() != nullptr; }

cudaError_t launch_stage1_ring(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    if (p.g_ring.empty()) return cudaSuccess;
    const int64_t nblocks = (int64_t)p.g_ring.size() * p.ring_nseg;
    if (nblocks > 0x7fffffff) return cudaErrorInvalidValue;
    if (stream_enabled() && p.nsamp <= 0x7fffffff && (p.ws_format == WS_PK16 || p.ws_format == WS_I32)) {
        CUtensorMap tm;
        cudaError_t e = make_input_map(p, d_in, kCG, kHalf, &tm, /*swizzle64=*/true);
        if (e != cudaSuccess) return e;
        int lds = 0;
        while ((1 << lds) < p.ds) ++lds;
        Stage1StreamFn fn = (p.ws_format == WS_PK16) ? pick_stream<WS_PK16>(p.cps) : pick_stream<WS_I32>(p.cps);
        if (!fn) return cudaErrorInvalidValue;
        fn<<<(unsigned)nblocks, kThreadsT, kSmemStream, st>>>(tm, p.d_s1, p.d_ws, p.ws_pitch, p.n1d, p.cps, p.ds, lds,
                                                             p.t2.M, p.d_g_ring, (int)p.g_ring.size(),
                                                             p.ring_seg_rows);
        return cudaPeekAtLastError();
    }
    Stage1RingFn fn = (p.ws_format == WS_PK16) ? pick_ring_nchan<WS_PK16>(p.nchan)
                    : (p.ws_format == WS_I32) ? pick_ring_nchan<WS_I32>(p.nchan) : nullptr;
    if (!fn) return cudaErrorInvalidValue;
    fn<<<(unsigned)nblocks, kThreadsR, kSmemRing, st>>>((const uint8_t *)d_in, p.d_s1, p.d_ws, p.ws_pitch,
                                                        p.n1d, p.nsamp, p.nchan, p.cps, p.ds, p.t2.M,
                                                        p.d_g_ring, (int)p.g_ring.size(), p.ring_seg_rows);
    return cudaPeekAtLastError();
}

}  // namespace gsp
