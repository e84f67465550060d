// gsp_stage1.cu — tiled stage-1 kernels (channel -> subband shift-and-sum + downsample).
//
//   S_s[t]  = sum_{c in subband s} x[t + s1[c]][c]      (Algorithm 1/2 of the paper applied per
//   S'_s[u] = sum_{k<ds} S_s[u*ds + k]   (un-divided)     subband: PAPER.md:104-166, sub-band
//                                                         method PAPER.md:100)
//
// The input is time-major (x[t][c], "numpts x numchan"), the sum runs along
// time-shifted columns.  One CTA owns 64 consecutive channels x kTileS consecutive S-samples:
//
//   load phase    every lane reads 4 channels x 4 rows (4 coalesced 32-bit loads; a warp request
//                 covers 4 rows x one full 32-byte sector), transposes the 4x4 bytes in registers
//                 (8 PRMT) and stores four words "one channel x 4 consecutive rows" into a
//                 CHANNEL-MAJOR shared tile.  Channel c's row of the tile starts at input row
//                 t0 + (s1[c] & ~127): the coarse part of the shift is applied by the store, so the
//                 tile is kTileS+128 samples long whatever the dispersion sweep H1 is.
//   gather phase  lanes take consecutive words of a channel row (bank-conflict free), the residual
//                 shift s1[c] & 127 is a word offset plus a funnel shift, and four samples per
//                 word are summed in two u16x2 accumulators (even / odd bytes; cps*255 < 2^16).
//   reduce/store  16-channel partial sums meet in shared memory, are folded over ds consecutive
//                 samples and written in the workspace format stage 2 reads.
//
// float32 input uses the same structure with one sample per word (no packing, no funnel shift).

#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "gsp_internal.h"

namespace gsp {

namespace {

constexpr int kTileS = 1024;                 // S-samples (before downsampling) per CTA tile
constexpr int kCG = 64;                      // channels per CTA
constexpr int kWinGran = 128;                // granularity of the per-channel window start (rows)
constexpr int kPitchW = (kTileS + kWinGran) / 4 + 1;   // 289 words per channel row (odd: the
                                                       // transposing stores hit 32 distinct banks)
constexpr int kThreads1 = 256;
constexpr int kSmem1 = kCG * kPitchW * 4;    // 73,984 bytes -> 3 CTAs per SM

// ---------------------------------------------------------------------------------------------
// uint8 input
// ---------------------------------------------------------------------------------------------
template <int FMT, int NCHAN>
__global__ void __launch_bounds__(kThreads1, 3)
stage1_tiled_u8_kernel(const uint8_t *__restrict__ x, const int32_t *__restrict__ s1,
                       void *__restrict__ ws, int64_t ws_pitch, int64_t n1d, int64_t nsamp, int nchan,
                       int cps, int ds, int M, const int32_t *__restrict__ glist, int ngroups) {
    extern __shared__ __align__(16) uint32_t xs[];   // [kCG][kPitchW]
    __shared__ int2 sh_g[kCG];                        // per channel: {word offset of its first gathered
                                                      // word, funnel shift in bits} (residual s1 & 127)

    const int group = __ldg(glist + blockIdx.x % ngroups);
    const int64_t tile = blockIdx.x / ngroups;
    const int64_t t0 = tile * kTileS;                 // first S-sample (= input row before shifting)
    const int cfirst = group * kCG;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x < kCG) {
        const int c = cfirst + threadIdx.x;
        const int e = (c < nchan) ? (__ldg(s1 + c) & (kWinGran - 1)) : 0;
        sh_g[threadIdx.x] = make_int2(threadIdx.x * kPitchW + (e >> 2), (e & 3) * 8);
    }

    // ------------------------------------ load + transpose ------------------------------------
    {
        const int col = warp >> 2, wi = warp & 3;     // 32-channel column, warp within the column
        const int qi = lane & 7, g = lane >> 3;       // channel quad, row group
        const int cl = col * 32 + 4 * qi;             // local channel of the quad's first byte
        const int c0 = cfirst + cl;
        const bool live = c0 < nchan;                 // nchan % 4 == 0: a quad is all in or all out
        int w128[4];
        int lo = INT32_MAX, hi = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            w128[k] = live ? (__ldg(s1 + c0 + k) & ~(kWinGran - 1)) : 0;
            if (live) {
                lo = min(lo, w128[k]);
                hi = max(hi, w128[k]);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        if (live) {                                   // (a dead quad exists only in a partial group)
            const int nblk = (hi - lo + kTileS + kWinGran + 4 + 15) >> 4;   // 16-row blocks
            int dw[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) dw[k] = (w128[k] - lo) >> 2;
            const int64_t rbase = t0 + lo + 4 * g;    // first row of this lane's 4-row blocks
            // With NCHAN known at compile time every load of an unrolled iteration is
            // [one 64-bit pointer + immediate]; NCHAN == 0 is the run-time fallback.
            const int64_t nc = NCHAN ? NCHAN : nchan;
            const uint8_t *src = x + rbase * nc + c0;
            uint32_t *dst = xs + cl * kPitchW;
            const bool inside = t0 + lo + 16 * (int64_t)nblk <= nsamp;   // column-uniform
            // rows (rel_blk*16 + i) below the pointer pb
            auto load_block = [&](const uint8_t *pb, int rel_blk, uint32_t (&v)[4]) {
#pragma unroll
                for (int i = 0; i < 4; ++i) v[i] = __ldg((const uint32_t *)(pb + (rel_blk * 16 + i) * nc));
            };
            auto load_block_checked = [&](int mb, uint32_t (&v)[4]) {
                const uint8_t *pb = src + (int64_t)mb * 16 * nc;
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    v[i] = (rbase + 16 * (int64_t)mb + i < nsamp) ? __ldg((const uint32_t *)(pb + i * nc)) : 0u;
            };
            auto store_block = [&](int mb, const uint32_t (&v)[4]) {
                // 4x4 byte transpose: v[i] = row i, bytes = channels -> o[k] = channel k, bytes = rows
                const uint32_t ta = __byte_perm(v[0], v[1], 0x5140), tb = __byte_perm(v[0], v[1], 0x7362);
                const uint32_t tc = __byte_perm(v[2], v[3], 0x5140), td = __byte_perm(v[2], v[3], 0x7362);
                uint32_t o[4];
                o[0] = __byte_perm(ta, tc, 0x5410);
                o[1] = __byte_perm(ta, tc, 0x7632);
                o[2] = __byte_perm(tb, td, 0x5410);
                o[3] = __byte_perm(tb, td, 0x7632);
                const int widx = 4 * mb + g;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int tw = widx - dw[k];
                    if ((unsigned)tw < (unsigned)kPitchW) dst[k * kPitchW + tw] = o[k];
                }
            };
            int mb = wi;
            if (inside) {
                // groups of four blocks (16 loads); the next group's loads are issued before the
                // current group is transposed and stored: up to 32 loads in flight per thread
                if (mb + 12 < nblk) {
                    const uint8_t *pb = src + (int64_t)mb * 16 * nc;
                    uint32_t a[4][4], b[4][4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) load_block(pb, 4 * j, a[j]);
                    for (;;) {
                        bool more = mb + 16 + 12 < nblk;
                        if (more) {
#pragma unroll
                            for (int j = 0; j < 4; ++j) load_block(pb, 16 + 4 * j, b[j]);
                        }
#pragma unroll
                        for (int j = 0; j < 4; ++j) store_block(mb + 4 * j, a[j]);
                        mb += 16;
                        pb += 256 * nc;
                        if (!more) break;
                        more = mb + 16 + 12 < nblk;
                        if (more) {
#pragma unroll
                            for (int j = 0; j < 4; ++j) load_block(pb, 16 + 4 * j, a[j]);
                        }
#pragma unroll
                        for (int j = 0; j < 4; ++j) store_block(mb + 4 * j, b[j]);
                        mb += 16;
                        pb += 256 * nc;
                        if (!more) break;
                    }
                }
                for (; mb < nblk; mb += 4) {
                    uint32_t v0[4];
                    load_block(src + (int64_t)mb * 16 * nc, 0, v0);
                    store_block(mb, v0);
                }
            } else {                                  // last tiles of the input: rows are checked
                for (; mb < nblk; mb += 4) {
                    uint32_t v0[4];
                    load_block_checked(mb, v0);
                    store_block(mb, v0);
                }
            }
        }
    }
    __syncthreads();

    // ------------------------------------------ gather ------------------------------------------
    // warp = (16-channel slice, 512-sample half); lane + 32 j = word of the half; a slot is the
    // part of a subband inside the slice (min(cps,16) channels).
    const int slot_ch = cps < 16 ? cps : 16;
    const int slots_per_slice = 16 / slot_ch;
    const int slice = warp >> 1, half = warp & 1;
    // results of every slot of this slice are kept in registers until all warps finished reading xs
    // (slots_per_slice <= 4 because cps >= 4)
    uint32_t res[4][8];
#pragma unroll
    for (int si = 0; si < 4; ++si) {
        uint32_t E[4] = {0u, 0u, 0u, 0u}, O[4] = {0u, 0u, 0u, 0u};
        const int cl0 = slice * 16 + si * slot_ch;
        if (si < slots_per_slice && cfirst + cl0 < nchan) {
            for (int j = 0; j < slot_ch; ++j) {
                const int2 ge = sh_g[cl0 + j];
                const uint32_t *row = xs + ge.x + half * 128 + lane;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t a = __funnelshift_r(row[32 * q], row[32 * q + 1], ge.y);
                    E[q] += __byte_perm(a, 0u, 0x4240);   // bytes 0 and 2 -> u16 lanes
                    O[q] += __byte_perm(a, 0u, 0x4341);   // bytes 1 and 3 -> u16 lanes
                }
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            // natural order: samples (4w, 4w+1) and (4w+2, 4w+3) as u16 pairs
            res[si][2 * q] = __byte_perm(E[q], O[q], 0x5410);
            res[si][2 * q + 1] = __byte_perm(E[q], O[q], 0x7632);
        }
    }
    __syncthreads();                                  // xs is dead: reuse it for the partial sums

    // part[slot][kTileS] as u16 (two words per gathered word)
    uint2 *part = (uint2 *)xs;
#pragma unroll
    for (int si = 0; si < 4; ++si) {
        const int slot = slice * slots_per_slice + si;
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (si < slots_per_slice)
                part[slot * (kTileS / 4) + half * 128 + lane + 32 * q] = make_uint2(res[si][2 * q], res[si][2 * q + 1]);
    }
    __syncthreads();

    // ------------------------------- slot reduce + downsample + store -------------------------------
    // part holds u16 pairs: one word = two consecutive S-samples of one slot.  A work item is the
    // max(1, ds/2) consecutive words of one output (ds >= 2) or of two outputs (ds == 1).
    const uint32_t *p32 = xs;
    const int nsb = kCG / cps;                        // subbands in this tile
    const int slots_per_sb = cps / slot_ch;
    const int gw = ds >= 2 ? ds / 2 : 1;
    const int items = (kTileS / 2) / gw;
    const int64_t u0 = t0 / ds;
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
    for (int sb = 0; sb < nsb; ++sb) {
        const int s = group * nsb + sb;
        if (s * cps >= nchan) break;
        for (int it = threadIdx.x; it < items; it += kThreads1) {
            uint32_t v0 = 0, v1 = 0;
            for (int sl = 0; sl < slots_per_sb; ++sl) {
                const uint32_t *pp = p32 + (sb * slots_per_sb + sl) * (kTileS / 2) + it * gw;
                for (int k = 0; k < gw; ++k) {
                    const uint32_t w = pp[k];
                    v0 += w & 0xffffu;
                    v1 += w >> 16;
                }
            }
            if (ds == 1) {
                emit(s, u0 + 2 * it, (int)v0);
                emit(s, u0 + 2 * it + 1, (int)v1);
            } else {
                emit(s, u0 + it, (int)(v0 + v1));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// One-stage plans (nsub == nchan: every channel is its own subband, s1 = 0, s2[d][c] = the one-stage
// delays — Algorithm 2 of the paper, which also moves the data to a channel-major
// layout).  Stage 1 is then a pure transposition (+ downsample): x[t][c] -> S'_c[u] in the
// format the tiled stage 2 reads, so the one-stage sum runs on the product stage-2 kernel.
// One CTA = 64 channels x 256 rows: coalesced 16-byte loads of the 64-byte row segments into a
// time-major shared tile (pitch 68 bytes = 17 words: byte-column reads are conflict-free), then every
// warp walks 8 channels with lanes on consecutive rows, folds ds rows with shuffles and stores.
// ---------------------------------------------------------------------------------------------
constexpr int kTrRows = 256;
constexpr int kTrPitch = 68;

template <int FMT>
__global__ void __launch_bounds__(256)
stage1_transpose_u8_kernel(const uint8_t *__restrict__ x, void *__restrict__ ws, int64_t ws_pitch, int64_t n1d,
                           int64_t nsamp, int nchan, int ds, int lds, int M) {
    __shared__ __align__(16) uint8_t tile[kTrRows * kTrPitch];
    const int ngroups = nchan / kCG;
    const int cfirst = (int)(blockIdx.x % ngroups) * kCG;
    const int64_t t0 = (int64_t)(blockIdx.x / ngroups) * kTrRows;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    {
        const int q = threadIdx.x & 3, r0 = threadIdx.x >> 2;          // 16-byte quarter of a row, row of a pass
#pragma unroll
        for (int pass = 0; pass < 4; ++pass) {
            const int r = r0 + 64 * pass;
            uint4 v = make_uint4(0u, 0u, 0u, 0u);
            if (t0 + r < nsamp) v = __ldg((const uint4 *)(x + (t0 + r) * (int64_t)nchan + cfirst) + q);
            uint32_t *d = (uint32_t *)(tile + r * kTrPitch + 16 * q);   // 68 r + 16 q: 4-byte aligned
            d[0] = v.x, d[1] = v.y, d[2] = v.z, d[3] = v.w;
        }
    }
    __syncthreads();
    for (int cc = 0; cc < 8; ++cc) {
        const int c = 8 * warp + cc;
#pragma unroll
        for (int j = 0; j < kTrRows / 32; ++j) {
            const int r = lane + 32 * j;
            int v = tile[r * kTrPitch + c];
            for (int o = 1; o < ds; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            const int64_t u = (t0 + r) >> lds;
            if ((r & (ds - 1)) == 0 && u < n1d) {
                if (FMT == WS_I32) {
                    ((int32_t *)ws)[(int64_t)(cfirst + c) * ws_pitch + u] = v;
                } else {  // WS_PK16: W[i] = S'[i] | S'[i+M] << 16
                    uint16_t *h = (uint16_t *)ws + 2 * ((int64_t)(cfirst + c) * ws_pitch);
                    h[2 * u] = (uint16_t)v;
                    if (u >= M) h[2 * (u - M) + 1] = (uint16_t)v;
                }
            }
        }
    }
}

}  // namespace

bool stage1_transpose_supported(const gsp_plan &p) {
    if (p.dtype != GSP_U8 || p.cps != 1 || p.nchan % kCG != 0) return false;
    return p.ds >= 1 && p.ds <= 32 && (p.ds & (p.ds - 1)) == 0;
}

cudaError_t launch_stage1_transpose(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    const int64_t total = p.n1d * (int64_t)p.ds;
    const int64_t ntile = (total + kTrRows - 1) / kTrRows;
    const int ngroups = p.nchan / kCG;
    if (ntile * ngroups > 0x7fffffff) return cudaErrorInvalidValue;
    int lds = 0;
    while ((1 << lds) < p.ds) ++lds;
    const unsigned grid = (unsigned)(ntile * ngroups);     // channel group fastest: resident CTAs read whole rows
    if (p.ws_format == WS_PK16)
        stage1_transpose_u8_kernel<WS_PK16><<<grid, 256, 0, st>>>((const uint8_t *)d_in, p.d_ws, p.ws_pitch, p.n1d,
                                                                  p.nsamp, p.nchan, p.ds, lds, p.t2.M);
    else if (p.ws_format == WS_I32)
        stage1_transpose_u8_kernel<WS_I32><<<grid, 256, 0, st>>>((const uint8_t *)d_in, p.d_ws, p.ws_pitch, p.n1d,
                                                                 p.nsamp, p.nchan, p.ds, lds, p.t2.M);
    else
        return cudaErrorInvalidValue;
    return cudaPeekAtLastError();
}

bool stage1_tiled_supported(const gsp_plan &p) {
    if (p.dtype != GSP_U8) return false;
    const int c = p.cps;
    if (!(c == 4 || c == 8 || c == 16 || c == 32 || c == 64)) return false;
    const int d = p.ds;
    if (d < 1 || d > 256 || (d & (d - 1))) return false;
    if ((int64_t)c * 255 > 65535) return false;
    return true;
}

typedef void (*Stage1Fn)(const uint8_t *, const int32_t *, void *, int64_t, int64_t, int64_t, int, int,
                         int, int, const int32_t *, int);

template <int FMT>
static Stage1Fn pick_stage1_nchan(int nchan) {
    switch (nchan) {  // common filterbank widths get immediate row offsets
        case 4096: return stage1_tiled_u8_kernel<FMT, 4096>;
        case 2048: return stage1_tiled_u8_kernel<FMT, 2048>;
        case 1024: return stage1_tiled_u8_kernel<FMT, 1024>;
        case 512: return stage1_tiled_u8_kernel<FMT, 512>;
        default: return stage1_tiled_u8_kernel<FMT, 0>;
    }
}

static Stage1Fn pick_stage1(const gsp_plan &p) {
    if (p.ws_format == WS_PK16) return pick_stage1_nchan<WS_PK16>(p.nchan);
    if (p.ws_format == WS_I32) return pick_stage1_nchan<WS_I32>(p.nchan);
    return nullptr;
}

cudaError_t configure_stage1(const gsp_plan &p) {
    if (!stage1_tiled_supported(p)) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute((const void *)pick_stage1_nchan<WS_I32>(p.nchan),
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem1);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute((const void *)pick_stage1_nchan<WS_PK16>(p.nchan),
                                cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem1);
}

cudaError_t launch_stage1_tiled(const gsp_plan &p, const void *d_in, const int32_t *d_groups, int ngroups,
                                cudaStream_t st) {
    if (ngroups <= 0) return cudaSuccess;
    const int64_t ntile = (p.n1d * p.ds + kTileS - 1) / kTileS;
    const int64_t nblocks = ntile * ngroups;
    if (nblocks > 0x7fffffff) return cudaErrorInvalidValue;
    Stage1Fn fn = pick_stage1(p);
    if (!fn) return cudaErrorInvalidValue;
    fn<<<(unsigned)nblocks, kThreads1, kSmem1, st>>>((const uint8_t *)d_in, p.d_s1, p.d_ws, p.ws_pitch,
                                                     p.n1d, p.nsamp, p.nchan, p.cps, p.ds, p.t2.M, d_groups, ngroups);
    return cudaPeekAtLastError();
}

}  // namespace gsp
