// gsp_stage1_f32.cu — tiled stage-1 kernel for float32 input.
//
//   S_s[t]  = sum_{c in subband s} x[t + s1[c]][c]      (Algorithm 1/2 of the paper applied per
//   S'_s[u] = sum_{k<ds} S_s[u*ds + k]   (un-divided)     subband: PAPER.md:104-166, sub-band
//                                                         method PAPER.md:100)
//
// The input is time-major, the sum runs down time-shifted columns.  With 4-byte elements the
// classic shared-memory transpose needs no register shuffling: a CTA owns one subband and
// kFT = 512 consecutive S-samples and walks the subband in passes of 16 channels.  Per pass
//
//   load    lanes = 16 channels x 2 rows: a warp request covers two full 64-byte row segments
//           (every byte of every sector used).  The rows read are the union of the 16 channels'
//           windows [t0 + s1[c], t0 + s1[c] + kFT); a lane stores its element DE-SKEWED, at
//           column (row - t0 - s1[c]) of its channel's row of the tile, and drops the rows
//           outside its own window (they are L2 hits of the neighbouring time tiles).
//           Sixteen loads per thread are in flight before the first store.
//           Channel rows start at a per-channel skew chosen so that the 32 lanes of a store hit
//           32 different banks whatever the shifts are: bank = 2*channel + row parity.
//   gather  the tile is already aligned in time: thread i adds column i of the 16 channel rows
//           (lanes on consecutive words: conflict-free), four columns per thread, accumulators in
//           registers across the passes.
//
// Epilogue: ds consecutive samples are folded with shuffles and stored as float32 S'.
// float32 sums are taken in float32 (reading A13 of DESIGN.md: <= 1e-5 of the row rms).
//
// That tile kernel is the fallback.  Plans whose shifts fit a shared-memory ring run the STREAMING kernels
// further down: stage1_f32_stream_kernel (one plan, clusters over the 16-channel groups of a subband) and, for the
// plans of one gsp_dedisperse_multi call, stage1_f32_shared_kernel + stage1_f32_combine[4]_kernel (one ring for
// all plans, group sums combined through a scratch array).

#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "gsp_internal.h"
#include "gsp_device.cuh"

namespace gsp {

namespace {

constexpr int kFT = 512;            // S-samples per CTA
constexpr int kFP = kFT + 32;       // tile row pitch in words (multiple of 32: the skew sets the bank)
constexpr int kFC = 16;             // channels per pass
constexpr int kFThreads = 128;
constexpr int kFU = 16;             // loads in flight per thread
constexpr int kFCols = kFT / kFThreads;

template <int NCHAN>
__global__ void __launch_bounds__(kFThreads)
stage1_f32_kernel(const float *__restrict__ x, const int32_t *__restrict__ s1, float *__restrict__ ws,
                  int64_t ws_pitch, int64_t n1d, int64_t nsamp, int nchan, int cps, int ds, int lds) {
    __shared__ float xs[kFC * kFP];
    __shared__ int sk[kFC];

    // subband fastest: the CTAs resident at one time cover whole input rows (DRAM page locality)
    const int s = blockIdx.x;
    const int64_t t0 = ((int64_t)blockIdx.z * gridDim.y + blockIdx.y) * kFT;
    if (t0 >= (n1d << lds)) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c16 = lane & 15, g = lane >> 4;
    const int64_t nc = NCHAN ? NCHAN : nchan;

    float acc[kFCols];
#pragma unroll
    for (int k = 0; k < kFCols; ++k) acc[k] = 0.f;

    const int npass = cps / kFC;
    for (int pass = 0; pass < npass; ++pass) {
        const int c = s * cps + pass * kFC + c16;
        const int sh = __ldg(s1 + c);
        int smin = sh, smax = sh;
#pragma unroll
        for (int o = 1; o < 16; o <<= 1) {
            smin = min(smin, __shfl_xor_sync(0xffffffffu, smin, o));
            smax = max(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        }
        const int skew = (2 * c16 + sh) & 31;
        if (tid < kFC) sk[c16] = skew;
        const int nrows = kFT + smax - smin;          // rows of the union window
        const int lead = sh - smin;                   // rows of the union before this channel's window
        const int64_t rbase = t0 + smin;
        const float *src = x + rbase * nc + c;
        float *dst = xs + c16 * kFP + skew - lead;    // element of union row rr goes to dst[rr]

        // this lane needs union rows [lo, lo + cnt): its own window, cut at the end of the input
        const int64_t left = nsamp - rbase;
        const int lim = left < (int64_t)nrows ? (int)left : nrows;
        const int lo = lead;
        const unsigned cnt = (unsigned)max(0, min(lead + kFT, lim) - lead);
        if (lim < lead + kFT) {                       // rows past the end of the input read as zero
            for (int i = tid >> 4; i < kFT; i += kFThreads / 16)
                if (i + lead >= lim) xs[c16 * kFP + skew + i] = 0.f;
        }
        for (int rr0 = 2 * warp + g; rr0 < nrows; rr0 += 8 * kFU) {
            const float *sp = src + (int64_t)rr0 * nc;
            float *dp = dst + rr0;
            const unsigned off = (unsigned)(rr0 - lo);
            float v[kFU];
#pragma unroll
            for (int k = 0; k < kFU; ++k)
                if (off + 8u * k < cnt) v[k] = __ldg(sp + (int64_t)(8 * k) * nc);
#pragma unroll
            for (int k = 0; k < kFU; ++k)
                if (off + 8u * k < cnt) dp[8 * k] = v[k];
        }
        __syncthreads();

#pragma unroll 4
        for (int j = 0; j < kFC; ++j) {
            const float *row = xs + j * kFP + sk[j] + tid;
#pragma unroll
            for (int k = 0; k < kFCols; ++k) acc[k] += row[kFThreads * k];
        }
        __syncthreads();
    }

    // ---- downsample (fold ds consecutive samples, held by consecutive lanes) + store
#pragma unroll
    for (int k = 0; k < kFCols; ++k) {
        const int i = tid + kFThreads * k;
        float v = acc[k];
        for (int o = 1; o < ds; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((i & (ds - 1)) == 0) {
            const int64_t u = (t0 + i) >> lds;
            if (u < n1d) ws[(int64_t)s * ws_pitch + u] = v;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Streaming variant (the one gsp_dedisperse runs when the shifts fit its ring): no transposition.
//
// A thread-block CLUSTER owns one subband and a segment of `seg` S-samples; CTA g of the cluster
// owns the subband's g-th 16-channel group.  Its producer warp streams boxes of 128 rows x 16
// channels (64-byte row segments, 8 KB) with 2-D tiled TMA loads into a ring of NS slots that stays
// TIME-MAJOR: ring[row][16].  The gather runs with lanes = (channel, output parity): lane (c, h)
// reads ring[t + 2j + h + s1[c]][c] for sixteen outputs j — its bank is 16*(row parity) + c, so a
// warp request is conflict-free whatever the per-channel shifts are — and the sixteen channel lanes
// are then summed with a transposing shuffle tree (15 shuffles for 16 outputs).  Every input
// element crosses shared memory once (TMA write + one LDS) and is read from DRAM once per segment
// plus the group's shift spread.  Eight consumer warps work independently: each waits on the full
// barriers of the slots its own rows live in and releases a slot (one arrive per warp) once its
// rows are behind it; there is no CTA-wide barrier in the loop.
// The group sums of a segment stay in the CTA's shared memory; after a cluster barrier CTA g adds
// the g-th part of the segment over all CTAs through distributed shared memory in a fixed order
// (deterministic: no float atomics), folds ds samples and stores S'.
// Why a cluster: the CTAs of a subband then run at the same time on neighbouring rows, and with the
// subband index fastest in the grid the resident CTAs read whole 16 KB input rows — measured 5.2
// TB/s against 2.7 TB/s when one CTA walked the four groups one after the other (DRAM page misses).
// ---------------------------------------------------------------------------------------------
constexpr int kSRows = 128;                      // rows per ring slot / TMA box
constexpr int kSSlotBytes = kSRows * kFC * 4;    // 8 KB
constexpr int kSWarps = 8;                       // consumer warps; warp 8 is the producer
constexpr int kSThreads = (kSWarps + 1) * 32;
constexpr int kSChunk = 32 * kSWarps;            // S-samples per chunk (32 per warp)

// Per-plan arguments of one launch: up to kMaxMulti plans (DM ranges with their own subband DM and
// downsampling) read the SAME input; their clusters sit next to each other in the grid, so the rows one
// of them pulls from DRAM are L2 hits for the others (gsp_dedisperse_multi).
constexpr int kMaxMulti = 4;
struct F32StreamArgs {
    const int32_t *s1[kMaxMulti];
    float *ws[kMaxMulti];
    int64_t ws_pitch[kMaxMulti];
    int64_t n1d[kMaxMulti];
    int ds[kMaxMulti];
    int lds[kMaxMulti];
    int np;
};

__global__ void __launch_bounds__(kSThreads, 3)
stage1_f32_stream_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ F32StreamArgs A, int cps,
                         int NS, int seg) {
    constexpr int UNR = 1;                                    // 32-output blocks per warp and chunk (2 measured slower)
    constexpr int CH = kSChunk * UNR;                         // S-samples per chunk
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(128) uint8_t smem_fs[];
    __shared__ float fold_scratch[8];
    uint64_t *full = (uint64_t *)smem_fs;                     // [NS <= 16] box landed
    uint64_t *empty = full + 16;                              // [NS <= 16] all consumer warps are past the slot
    const float *ring = (const float *)(smem_fs + 256);       // [NS][128 rows][16 channels]
    float *outs = (float *)(smem_fs + 256 + NS * kSSlotBytes);   // [seg] this group's sums

    // cluster = the 16-channel groups of one subband (cluster rank = group), subband fastest in the
    // grid: the CTAs resident at one time read whole input rows (DRAM page locality)
    const int ngroups = cps / kFC;
    const int g = (int)cluster.block_rank();
    const int cl = blockIdx.x / ngroups;                      // cluster index = subband * np + plan
    const int pl = cl % A.np, s = cl / A.np;
    const int32_t *__restrict__ s1 = A.s1[pl];
    float *__restrict__ ws = A.ws[pl];
    const int64_t ws_pitch = A.ws_pitch[pl], n1d = A.n1d[pl];
    const int ds = A.ds[pl], lds = A.lds[pl];
    const int64_t tseg = (int64_t)blockIdx.y * seg;     // seg: S-samples per CTA segment
    const int64_t total = n1d << lds;
    if (tseg >= total) return;                                // (a shorter plan of a multi-plan launch: the whole cluster leaves)
    const int segn = (int)((total - tseg < seg) ? (total - tseg) : seg);
    const int nk = (segn + CH - 1) / CH;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int c16 = lane & 15, h = lane >> 4;

    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], kSWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int c0 = s * cps + g * kFC;
    const int sh = __ldg(s1 + c0 + c16);
    int smin = sh, smax = sh;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        smin = min(smin, __shfl_xor_sync(0xffffffffu, smin, o));
        smax = max(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    }
    const int spread = smax - smin;
    const int nslot = (CH * nk + spread + kSRows - 1) / kSRows;

    if (warp == kSWarps) {
        // ------------------------------------ producer ------------------------------------
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            const int64_t rbase = tseg + smin;
            for (int j = 0; j < nslot; ++j) {
                while (!mbar_try_wait(&empty[st], ph ^ 1u)) __nanosleep(64);
                mbar_arrive_expect_tx(&full[st], kSSlotBytes);
                tma_load_2d((void *)(smem_fs + 256 + st * kSSlotBytes), &tmap, c0, (int)(rbase + (int64_t)kSRows * j),
                            &full[st]);
                if (++st == NS) {
                    st = 0;
                    ph ^= 1u;
                }
            }
        }
        __syncwarp();
    } else {
        // ------------------------------------ consumers ------------------------------------
        // slot indices: full barriers passed (have) / slots released by this warp (rel), with their ring
        // slot and phase kept incrementally (NS need not be a power of two)
        int have = 0, hslot = 0, rslot = 0;
        uint32_t hph = 0;
        auto wait_upto = [&](int idx) {   // every slot up to idx (inclusive) has landed
            while (have <= idx) {
                mbar_wait(&full[hslot], hph);
                ++have;
                if (++hslot == NS) {
                    hslot = 0;
                    hph ^= 1u;
                }
            }
        };
        const uint32_t ringw = (uint32_t)(NS * kSRows * kFC);   // ring size in floats
        uint32_t xoff[16];                                      // ring offset of output (j ^ c16): 2 rows per output
#pragma unroll
        for (int j = 0; j < 16; ++j) xoff[j] = 2u * kFC * (uint32_t)(j ^ c16);
        uint32_t abase = (uint32_t)((32 * UNR * warp + h + (sh - smin)) * kFC + c16) % ringw;   // chunk 0
        for (int k = 0; k < nk; ++k) {
            const int r0 = CH * k + 32 * UNR * warp;          // first ring row the warp touches
            // the slots this warp's rows live in — and, so that it may hand them back below, the chunk's own
            // slots: a slot is only released after its box was seen landed (the box was then issued, which
            // needed every warp's release of the slot's previous use: an arrive cannot land in the wrong phase)
            wait_upto(max((r0 + 32 * UNR - 1 + spread) >> 7, (CH / kSRows) * (k + 1) - 1));
            // ring[(row of output r0 + 32u + 2j + h, channel c16)], wrapping at the end of the ring.
            // Register j holds output (j ^ c16): with this lane-dependent order the transposing sum below
            // needs no selects (every lane keeps its low registers and sends its high ones)
            float v[UNR][16];
            if (__all_sync(0xffffffffu, abase + 2u * kFC * (16u * UNR - 1u) < ringw)) {   // no lane wraps in this chunk
                const float *rp = ring + abase;
#pragma unroll
                for (int u = 0; u < UNR; ++u)
#pragma unroll
                    for (int j = 0; j < 16; ++j) v[u][j] = rp[32 * kFC * u + xoff[j]];
            } else {
#pragma unroll
                for (int u = 0; u < UNR; ++u)
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        uint32_t a = abase + 32u * kFC * u + xoff[j];
                        a = (a >= ringw) ? a - ringw : a;
                        v[u][j] = ring[a];
                    }
            }
            abase += (uint32_t)(CH * kFC);
            abase = (abase >= ringw) ? abase - ringw : abase;
            // transposing sum over the 16 channel lanes: at level m the partner (lane ^ m) holds in its
            // register j + m the output this lane holds in register j; lane c16 ends with output c16
#pragma unroll
            for (int m = 8; m >= 1; m >>= 1) {
#pragma unroll
                for (int j = 0; j < m; ++j)
#pragma unroll
                    for (int u = 0; u < UNR; ++u) v[u][j] += __shfl_xor_sync(0xffffffffu, v[u][j + m], m);
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) outs[r0 + 32 * u + 2 * c16 + h] = v[u][0];
            // this warp is past chunk k: it gives the chunk's slots back (one arrive per warp and slot; the
            // producer refills a slot when all eight warps have) — no CTA barrier in the loop
            __syncwarp();
#pragma unroll
            for (int q = 0; q < CH / kSRows; ++q) {
                if (lane == 0 && (CH / kSRows) * k + q < nslot) mbar_arrive(&empty[rslot]);
                if (++rslot == NS) rslot = 0;
            }
        }
    }

    // ---- sum the groups (fixed order: deterministic), fold ds samples, store: CTA g takes the g-th
    //      part of the segment and reads the other CTAs' sums through distributed shared memory
    cluster_sync_publish();
    {
        const int part = seg / ngroups;
        const float *src[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) src[r] = cluster.map_shared_rank(outs, r < ngroups ? r : 0);
        for (int i0 = g * part; i0 < (g + 1) * part; i0 += kSWarps * 32) {
            const int i = i0 + (int)threadIdx.x;
            if (threadIdx.x < kSWarps * 32) {
                float r = 0.f;
#pragma unroll
                for (int q = 0; q < 8; ++q)
                    if (q < ngroups) r += src[q][i];
                r = fold_ds256(r, ds, (int)threadIdx.x, fold_scratch, 2);
                if ((i & (ds - 1)) == 0) {
                    const int64_t u = (tseg + i) >> lds;
                    if (i < segn && u < n1d) ws[(int64_t)s * ws_pitch + u] = r;
                }
            }
        }
    }
    cluster_sync_relaxed();   // remote reads are done before any CTA of the cluster exits
}


// ---------------------------------------------------------------------------------------------
// Shared ring for several plans (gsp_dedisperse_multi: the DM ranges of a DDplan over one float32
// input, each with its own subband DM, i.e. its own shifts).  One CTA owns one 16-channel group and a
// segment of S-samples and streams the group's rows ONCE through the time-major ring of the kernel
// above; every plan then gathers from the same slots with its own shifts (same lanes = channels
// gather, same transposing shuffle tree: a group's partial sums are bit-identical to the single-plan
// kernel's).  What makes one ring enough although the plans' shifts differ by thousands of rows: plan
// p works `lag_p` chunks behind the stream head — in iteration i it produces chunk i - lag_p, where
// lag_p = (smin_p - min_q smin_q) / 256 — so that all plans read the rows just behind the head and
// the ring spans one chunk plus the largest shift spread, not the difference between the plans.
// The plans' output chunks of one iteration therefore differ, and so do the groups' of a subband
// (their smin differ): the group sums cannot meet in shared memory.  Each CTA writes its group's
// partial sums to a plan-owned scratch array P[group][t] (coalesced), and stage1_f32_combine_kernel
// adds the groups of a subband in the fixed order 0, 1, ... (the order of the cluster kernel), folds
// ds samples and stores S'.  Results are bit-identical to separate gsp_dedisperse calls.
// ---------------------------------------------------------------------------------------------
struct F32SharedArgs {
    const int32_t *s1[kMaxMulti];
    float *part[kMaxMulti];          // [nchan / 16][part_pitch] partial sums of the 16-channel groups
    int64_t total[kMaxMulti];        // S-samples that feed an output (n1d << lds)
    int64_t part_pitch;
};

template <int NP>
__global__ void __launch_bounds__(kSThreads, 2)
stage1_f32_shared_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ F32SharedArgs A, int NS,
                         int seg) {
    constexpr int CH = kSChunk;                               // S-samples per chunk and iteration
    extern __shared__ __align__(128) uint8_t smem_fs[];
    uint64_t *full = (uint64_t *)smem_fs;                     // [NS <= 16] box landed
    uint64_t *empty = full + 16;                              // [NS <= 16] all consumer warps are past the slot
    const float *ring = (const float *)(smem_fs + 256);       // [NS][128 rows][16 channels]

    const int G = blockIdx.x;                                 // 16-channel group (fastest: resident CTAs read whole rows)
    const int64_t tseg = (int64_t)blockIdx.y * seg;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int c16 = lane & 15, h = lane >> 4;

    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], kSWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // per plan: this lane's shift, the group's smallest / largest shift, chunks in this segment
    const int c0 = G * kFC;
    int sh[NP], smin[NP], spread[NP], nk[NP];
    int smin_all = 0x7fffffff;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        sh[p] = __ldg(A.s1[p] + c0 + c16);
        int lo = sh[p], hi = sh[p];
#pragma unroll
        for (int o = 1; o < 16; o <<= 1) {
            lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        smin[p] = lo;
        spread[p] = hi - lo;
        const int64_t left = A.total[p] - tseg;
        nk[p] = left <= 0 ? 0 : (int)((min(left, (int64_t)seg) + CH - 1) / CH);
        smin_all = min(smin_all, lo);
    }
    int lag[NP], rel[NP], span = 0, NI = 0;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const int D = smin[p] - smin_all;
        lag[p] = D / CH;
        rel[p] = sh[p] - smin_all - CH * lag[p];              // this lane's row offset inside the iteration's window
        span = max(span, D - CH * lag[p] + spread[p]);        // rows past the chunk the window reaches
        if (nk[p] > 0) NI = max(NI, nk[p] + lag[p]);
    }
    if (NI == 0) return;
    const int nslot = (CH * NI + span + kSRows - 1) / kSRows;

    if (warp == kSWarps) {
        // ------------------------------------ producer ------------------------------------
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            const int64_t rbase = tseg + smin_all;
            for (int j = 0; j < nslot; ++j) {
                while (!mbar_try_wait(&empty[st], ph ^ 1u)) __nanosleep(64);
                mbar_arrive_expect_tx(&full[st], kSSlotBytes);
                tma_load_2d((void *)(smem_fs + 256 + st * kSSlotBytes), &tmap, c0, (int)(rbase + (int64_t)kSRows * j),
                            &full[st]);
                if (++st == NS) {
                    st = 0;
                    ph ^= 1u;
                }
            }
        }
        return;
    }

    // ------------------------------------ consumers ------------------------------------
    int have = 0, hslot = 0, rslot = 0;
    uint32_t hph = 0;
    auto wait_upto = [&](int idx) {   // every slot up to idx (inclusive) has landed
        while (have <= idx) {
            mbar_wait(&full[hslot], hph);
            ++have;
            if (++hslot == NS) {
                hslot = 0;
                hph ^= 1u;
            }
        }
    };
    // byte addresses in the shared window: one add per load
    const uint32_t ringb = (uint32_t)(NS * kSSlotBytes);      // ring size in bytes
    const uint32_t ring0 = smem_u32(ring);
    uint32_t xoff[16];                                        // byte offset of output (j ^ c16): 2 rows per output
#pragma unroll
    for (int j = 0; j < 16; ++j) xoff[j] = 4u * 2u * kFC * (uint32_t)(j ^ c16);
    uint32_t abase[NP];                                       // ring byte offset of the lane's first element, iteration 0
    float *outp[NP];                                          // where the lane's output of the current iteration goes
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        abase[p] = (4u * (uint32_t)((32 * warp + h + rel[p]) * kFC + c16)) % ringb;
        outp[p] = A.part[p] + ((int64_t)G * A.part_pitch + tseg + 32 * warp + 2 * c16 + h) - (int64_t)CH * lag[p];
    }
    auto lds_f32 = [](uint32_t addr) {
        float v;
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
        return v;
    };

    for (int i = 0; i < NI; ++i) {
        const int r0 = CH * i + 32 * warp;                    // first ring row of the iteration's window the warp touches
        // the slots the window of any plan can reach — and the iteration's own two slots, which the warp hands
        // back below (a slot is only released after its box was seen landed, see the kernel above)
        wait_upto(max((r0 + 31 + span) >> 7, (CH / kSRows) * (i + 1) - 1));
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const int k = i - lag[p];                         // the chunk plan p produces now (warp-uniform)
            if (k >= 0 && k < nk[p]) {
                float v[16];
                if (__all_sync(0xffffffffu, abase[p] + 4u * 2u * kFC * 15u < ringb)) {   // no lane wraps in this chunk
                    const uint32_t rp = ring0 + abase[p];
#pragma unroll
                    for (int j = 0; j < 16; ++j) v[j] = lds_f32(rp + xoff[j]);
                } else {
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        uint32_t a = abase[p] + xoff[j];
                        a = (a >= ringb) ? a - ringb : a;
                        v[j] = lds_f32(ring0 + a);
                    }
                }
                // transposing sum over the 16 channel lanes (same tree as the single-plan kernel)
#pragma unroll
                for (int m = 8; m >= 1; m >>= 1) {
#pragma unroll
                    for (int j = 0; j < m; ++j) v[j] += __shfl_xor_sync(0xffffffffu, v[j + m], m);
                }
                *outp[p] = v[0];
            }
            outp[p] += CH;
            abase[p] += (uint32_t)(CH * kFC * 4);
            abase[p] = (abase[p] >= ringb) ? abase[p] - ringb : abase[p];
        }
        __syncwarp();
#pragma unroll
        for (int q = 0; q < CH / kSRows; ++q) {
            if (lane == 0 && (CH / kSRows) * i + q < nslot) mbar_arrive(&empty[rslot]);
            if (++rslot == NS) rslot = 0;
        }
    }
}

// S'_s[u] = fold_ds( sum over the subband's groups, in the order 0, 1, ..., of P[group][t] ): the second half of
// the shared-ring path.  One thread per S-sample; 256-thread blocks start on multiples of 256 samples, as the
// cluster kernel's epilogue does, so the fold adds the same samples in the same order.
__global__ void __launch_bounds__(256)
stage1_f32_combine_kernel(const float *__restrict__ part, int64_t part_pitch, float *__restrict__ ws, int64_t ws_pitch,
                          int64_t n1d, int ngroups, int ds, int lds) {
    __shared__ float fold_scratch[8];
    const int s = blockIdx.y;
    const int64_t t = (int64_t)blockIdx.x * 256 + threadIdx.x;
    const int64_t total = n1d << lds;
    float r = 0.f;
    if (t < total)
        for (int q = 0; q < ngroups; ++q) r += part[((int64_t)s * ngroups + q) * part_pitch + t];
    r = fold_ds256(r, ds, (int)threadIdx.x, fold_scratch, 2);
    if ((threadIdx.x & (ds - 1)) == 0) {
        const int64_t u = t >> lds;
        if (t < total && u < n1d) ws[(int64_t)s * ws_pitch + u] = r;
    }
}


// The same for ds <= 32 and all plans of a call in one launch (blockIdx.z = plan), four consecutive S-samples per
// thread (16-byte loads).  The fold is the same perfect tree over consecutive samples as fold_ds256's butterfly:
// (x0 + x1) + (x2 + x3) inside the thread are its first two levels, the lanes continue with xor 1, 2, 4.
struct F32CombineArgs {
    const float *part[kMaxMulti];
    float *ws[kMaxMulti];
    int64_t ws_pitch[kMaxMulti], n1d[kMaxMulti];
    int ds[kMaxMulti], lds[kMaxMulti];
    int64_t part_pitch;
    int ngroups;
};

__global__ void __launch_bounds__(256)
stage1_f32_combine4_kernel(const __grid_constant__ F32CombineArgs A) {
    const int p = blockIdx.z, s = blockIdx.y;
    const int ds = A.ds[p], lds = A.lds[p];
    const int64_t n1d = A.n1d[p], total = n1d << lds;
    const int64_t t = ((int64_t)blockIdx.x * 256 + threadIdx.x) * 4;
    if ((int64_t)blockIdx.x * 1024 >= total) return;          // (CTA-uniform)
    float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
    if (t < total) {                                          // total is a multiple of ds; rows are padded to the segment
        const float *src = A.part[p] + (int64_t)s * A.ngroups * A.part_pitch + t;
        for (int q = 0; q < A.ngroups; ++q) {
            const float4 v = __ldg((const float4 *)(src + (int64_t)q * A.part_pitch));
            r.x += v.x, r.y += v.y, r.z += v.z, r.w += v.w;
        }
    }
    float *dst = A.ws[p] + (int64_t)s * A.ws_pitch[p];
    if (ds == 1) {
        if (t + 3 < n1d) {
            *(float4 *)(dst + t) = r;
        } else {
            if (t < n1d) dst[t] = r.x;
            if (t + 1 < n1d) dst[t + 1] = r.y;
            if (t + 2 < n1d) dst[t + 2] = r.z;
        }
        return;
    }
    const float a = r.x + r.y, b = r.z + r.w;
    if (ds == 2) {
        const int64_t u = t >> 1;
        if (u < n1d) dst[u] = a;
        if (u + 1 < n1d) dst[u + 1] = b;
        return;
    }
    float v = a + b;
    for (int o = 1; o < (ds >> 2); o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & ((ds >> 2) - 1)) == 0) {
        const int64_t u = t >> lds;
        if (u < n1d) dst[u] = v;
    }
}

}  // namespace

static bool tile_kernel_ok(const gsp_plan &p) {
    if (p.dtype != GSP_F32) return false;
    if (p.cps % kFC != 0) return false;
    const int d = p.ds;
    return d >= 1 && d <= 32 && (d & (d - 1)) == 0;   // (the tile kernel folds with shuffles only)
}

bool stage1_f32_supported(const gsp_plan &p) { return tile_kernel_ok(p) || p.f32_slots > 0; }

// Ring slots of the streaming kernel for this plan: 8 or 16, or 0 when the largest shift spread of a
// 16-channel group does not fit (the tile kernel runs instead).
static int stream_slots(const gsp_plan &p) {
    if (p.dtype != GSP_F32 || p.cps % kFC != 0 || p.ds < 1 || p.ds > 256 || (p.ds & (p.ds - 1))) return 0;
    if (!tma_available()) return 0;
    if (p.nsamp > 0x7fffffff) return 0;
    const int ng = p.cps / kFC;
    if (!(ng == 1 || ng == 2 || ng == 4 || ng == 8)) return 0;   // one cluster = the groups of a subband
    int spread = 0;
    for (int c0 = 0; c0 + kFC <= p.nchan; c0 += kFC) {
        const auto mm = std::minmax_element(p.s1.begin() + c0, p.s1.begin() + c0 + kFC);
        spread = std::max(spread, *mm.second - *mm.first);
    }
    // slots a warp's chunk can span + the lag of the slowest warp + two boxes of prefetch
    const int ns = (kSChunk + spread + 2 * kSRows - 1) / kSRows + 1 + 2;
    if (ns > 16) return 0;
    return ns < 10 ? 10 : ns;     // up to 10 slots fit two CTAs per SM with the long segment: spend them on prefetch
}

// decided once, at plan creation (gsp_plan_create calls this after the tables are built)
void plan_stage1_f32(gsp_plan &p) { p.f32_slots = stream_slots(p); }

bool stage1_f32_streams(const gsp_plan &p) { return p.f32_slots > 0; }

typedef void (*Stage1F32StreamFn)(const CUtensorMap, const F32StreamArgs, int, int, int);

// S-samples per CTA segment: long (less warm-up per byte) when two CTAs still fit an SM
static int stream_seg(int ns) { return ns <= 10 ? 8192 : 4096; }
static size_t stream_smem(int ns) { return 256 + (size_t)ns * kSSlotBytes + (size_t)stream_seg(ns) * 4; }

typedef void (*Stage1F32SharedFn)(const CUtensorMap, const F32SharedArgs, int, int);
constexpr int kSharedMaxSlots = 13;              // 13 slots = 104 KB: two CTAs per SM

static Stage1F32SharedFn pick_shared(int np) {
    switch (np) {
        case 2: return (Stage1F32SharedFn)stage1_f32_shared_kernel<2>;
        case 3: return (Stage1F32SharedFn)stage1_f32_shared_kernel<3>;
        case 4: return (Stage1F32SharedFn)stage1_f32_shared_kernel<4>;
        default: return nullptr;
    }
}

cudaError_t configure_stage1_f32(const gsp_plan &p) {
    if (p.dtype != GSP_F32) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute((const void *)(Stage1F32StreamFn)stage1_f32_stream_kernel,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stream_smem(16));
    for (int np = 2; np <= kMaxMulti && e == cudaSuccess; ++np)
        e = cudaFuncSetAttribute((const void *)pick_shared(np), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)(256 + kSharedMaxSlots * kSSlotBytes));
    return e;
}

// Plans that can share one streaming launch: same input geometry, every one of them streams.
bool stage1_f32_multi_ok(gsp_plan *const *plans, int np) {
    if (np < 1 || np > kMaxMulti) return false;
    for (int i = 0; i < np; ++i) {
        const gsp_plan &q = *plans[i], &p0 = *plans[0];
        if (q.f32_slots == 0) return false;
        if (q.nchan != p0.nchan || q.nsamp != p0.nsamp || q.nsub != p0.nsub || q.ws_format != WS_F32) return false;
    }
    return true;
}

// Ring slots the shared-ring kernel needs for these plans (0: more than two CTAs per SM can hold — the side by
// side launch of the cluster kernel runs instead).  Mirrors the kernel's own arithmetic, per 16-channel group.
static int shared_slots(gsp_plan *const *plans, int np) {
    const gsp_plan &p0 = *plans[0];
    int span = 0;
    for (int c0 = 0; c0 + kFC <= p0.nchan; c0 += kFC) {
        int smin[kMaxMulti], spread[kMaxMulti], smin_all = INT32_MAX;
        for (int i = 0; i < np; ++i) {
            const auto mm = std::minmax_element(plans[i]->s1.begin() + c0, plans[i]->s1.begin() + c0 + kFC);
            smin[i] = *mm.first;
            spread[i] = *mm.second - *mm.first;
            smin_all = std::min(smin_all, smin[i]);
        }
        for (int i = 0; i < np; ++i) span = std::max(span, (smin[i] - smin_all) % kSChunk + spread[i]);
    }
    const int ns = (kSChunk + span + 2 * kSRows - 1) / kSRows + 1 + 2;
    return ns <= kSharedMaxSlots ? std::max(ns, 10) : 0;
}

constexpr int kSharedSeg = 32768;   // S-samples per CTA segment of the shared-ring kernel (no per-segment buffer)

// Partial-sum scratch of the shared-ring path: nchan/16 rows of float32 per plan.  The row pitch depends on the
// plan's own input length only (n1d*ds <= nsamp, and plans that share a ring have the same nsamp), never on
// which plans happen to be grouped, so one allocation serves every grouping.
static int64_t shared_part_pitch(const gsp_plan &p) { return (p.nsamp + kSharedSeg - 1) / kSharedSeg * kSharedSeg; }

cudaError_t reserve_stage1_f32_shared(gsp_plan &q) {
    if (q.dtype != GSP_F32 || !stage1_f32_streams(q)) return cudaSuccess;   // never on the shared-ring path
    const size_t need = (size_t)(q.nchan / kFC) * (size_t)shared_part_pitch(q) * sizeof(float);
    if (q.d_f32_part && q.f32_part_bytes >= need) return cudaSuccess;
    if (q.d_f32_part) cudaFree(q.d_f32_part);
    q.d_f32_part = nullptr;
    q.f32_part_bytes = 0;
    cudaError_t e = cudaMalloc((void **)&q.d_f32_part, need);
    if (e != cudaSuccess) return e;
    q.f32_part_bytes = need;
    return cudaSuccess;
}

// Several plans on ONE ring: stage1_f32_shared_kernel into the plans' partial-sum scratch, then one combine
// launch per plan.  The scratch is reserved by gsp_plan_reserve_multi, else on first use here; when it cannot be
// had the caller (launch_stage1_f32_multi) runs the side-by-side launch instead.
static cudaError_t launch_stage1_f32_shared(gsp_plan *const *plans, int np, int ns, const void *d_in,
                                            cudaStream_t st) {
    const gsp_plan &p0 = *plans[0];
    int64_t total = 0;
    for (int i = 0; i < np; ++i) total = std::max<int64_t>(total, plans[i]->n1d * (int64_t)plans[i]->ds);
    const int64_t nseg = (total + kSharedSeg - 1) / kSharedSeg;
    if (nseg > 65535) return cudaErrorInvalidValue;
    const int64_t pitch = shared_part_pitch(p0);
    const int ngroups_all = p0.nchan / kFC;
    F32SharedArgs A = {};
    A.part_pitch = pitch;
    for (int i = 0; i < np; ++i) {
        gsp_plan &q = *plans[i];
        cudaError_t e = reserve_stage1_f32_shared(q);
        if (e != cudaSuccess) return e;
        A.s1[i] = q.d_s1;
        A.part[i] = q.d_f32_part;
        A.total[i] = q.n1d * (int64_t)q.ds;
    }
    const CUtensorMap *tm = nullptr;
    cudaError_t e = input_map(p0, TMAP_F32, d_in, kFC, kSRows, /*swizzle_bytes=*/0, &tm);
    if (e != cudaSuccess) return e;
    Stage1F32SharedFn fn = pick_shared(np);
    if (!fn) return cudaErrorInvalidValue;
    const size_t smem = 256 + (size_t)ns * kSSlotBytes;
    fn<<<dim3((unsigned)ngroups_all, (unsigned)nseg), kSThreads, smem, st>>>(*tm, A, ns, kSharedSeg);
    e = cudaPeekAtLastError();
    if (e != cudaSuccess) return e;
    bool small_ds = true;
    for (int i = 0; i < np; ++i) small_ds = small_ds && plans[i]->ds <= 32 && (plans[i]->ws_pitch % 4) == 0;
    if (small_ds) {                              // one launch for all plans, four samples per thread
        F32CombineArgs C = {};
        C.part_pitch = pitch;
        C.ngroups = p0.cps / kFC;
        for (int i = 0; i < np; ++i) {
            const gsp_plan &q = *plans[i];
            int lds = 0;
            while ((1 << lds) < q.ds) ++lds;
            C.part[i] = q.d_f32_part;
            C.ws[i] = (float *)q.d_ws;
            C.ws_pitch[i] = q.ws_pitch;
            C.n1d[i] = q.n1d;
            C.ds[i] = q.ds;
            C.lds[i] = lds;
        }
        stage1_f32_combine4_kernel<<<dim3((unsigned)((total + 1023) / 1024), (unsigned)p0.nsub, (unsigned)np), 256, 0,
                                     st>>>(C);
        return cudaPeekAtLastError();
    }
    for (int i = 0; i < np && e == cudaSuccess; ++i) {
        const gsp_plan &q = *plans[i];
        int lds = 0;
        while ((1 << lds) < q.ds) ++lds;
        const int64_t tot = q.n1d * (int64_t)q.ds;
        stage1_f32_combine_kernel<<<dim3((unsigned)((tot + 255) / 256), (unsigned)q.nsub), 256, 0, st>>>(
            q.d_f32_part, pitch, (float *)q.d_ws, q.ws_pitch, q.n1d, q.cps / kFC, q.ds, lds);
        e = cudaPeekAtLastError();
    }
    return e;
}

// One launch of the streaming kernel for np plans over the same input (np = 1: the plain case).  Two or more
// plans share ONE ring when their shift spreads allow (launch_stage1_f32_shared); otherwise their clusters sit
// side by side in the grid of the single-plan kernel.
cudaError_t launch_stage1_f32_multi(gsp_plan *const *plans, int np, const void *d_in, cudaStream_t st) {
    if (!stage1_f32_multi_ok(plans, np)) return cudaErrorInvalidValue;
    if (np >= 2) {
        const int nss = shared_slots(plans, np);
        if (nss > 0) {
            const cudaError_t es = launch_stage1_f32_shared(plans, np, nss, d_in, st);
            if (es != cudaErrorMemoryAllocation) return es;
            cudaGetLastError();   // no room for the partial-sum scratch: the side-by-side launch needs none
        }
    }
    const gsp_plan &p0 = *plans[0];
    F32StreamArgs A = {};
    A.np = np;
    int ns = 0;
    for (int i = 0; i < np; ++i) ns = std::max(ns, plans[i]->f32_slots);
    const int seg = stream_seg(ns);
    int64_t nseg = 0;
    for (int i = 0; i < np; ++i) {
        const gsp_plan &q = *plans[i];
        int lds = 0;
        while ((1 << lds) < q.ds) ++lds;
        A.s1[i] = q.d_s1;
        A.ws[i] = (float *)q.d_ws;
        A.ws_pitch[i] = q.ws_pitch;
        A.n1d[i] = q.n1d;
        A.ds[i] = q.ds;
        A.lds[i] = lds;
        nseg = std::max<int64_t>(nseg, (q.n1d * (int64_t)q.ds + seg - 1) / seg);
    }
    if (nseg > 65535) return cudaErrorInvalidValue;
    const CUtensorMap *tm = nullptr;
    cudaError_t e = input_map(p0, TMAP_F32, d_in, kFC, kSRows, /*swizzle_bytes=*/0, &tm);
    if (e != cudaSuccess) return e;
    const int ng = p0.cps / kFC;
    Stage1F32StreamFn fn = (Stage1F32StreamFn)stage1_f32_stream_kernel;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(p0.nsub * np * ng), (unsigned)nseg);
    cfg.blockDim = dim3(kSThreads);
    cfg.dynamicSmemBytes = stream_smem(ns);
    cfg.stream = st;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = (unsigned)ng;
    attr.val.clusterDim.y = 1;
    attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, fn, *tm, A, p0.cps, ns, seg);
    return e != cudaSuccess ? e : cudaPeekAtLastError();
}

// Kernels launch_stage1_f32_multi enqueues for these plans (gsp_dedisperse_multi_launches).
int stage1_f32_multi_launches(gsp_plan *const *plans, int np) {
    if (np < 2 || shared_slots(plans, np) == 0) return 1;          // side by side: one launch
    bool small_ds = true;
    for (int i = 0; i < np; ++i) small_ds = small_ds && plans[i]->ds <= 32 && (plans[i]->ws_pitch % 4) == 0;
    return 1 + (small_ds ? 1 : np);                                // shared ring + combine
}

cudaError_t launch_stage1_f32(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    const int64_t total = p.n1d * (int64_t)p.ds;
    int lds = 0;
    while ((1 << lds) < p.ds) ++lds;
    if (p.f32_slots) {
        gsp_plan *one = const_cast<gsp_plan *>(&p);
        return launch_stage1_f32_multi(&one, 1, d_in, st);
    }
    const int64_t ntile = (total + kFT - 1) / kFT;
    const int64_t ty = std::min<int64_t>(ntile, 32768), tz = (ntile + ty - 1) / ty;
    if (tz > 65535) return cudaErrorInvalidValue;
    dim3 grid((unsigned)p.nsub, (unsigned)ty, (unsigned)tz);
#define GSP_S1F(N)                                                                                     \
    stage1_f32_kernel<N><<<grid, kFThreads, 0, st>>>((const float *)d_in, p.d_s1, (float *)p.d_ws,     \
                                                     p.ws_pitch, p.n1d, p.nsamp, p.nchan, p.cps, p.ds, lds)
    switch (p.nchan) {  // common filterbank widths get immediate row offsets
        case 4096: GSP_S1F(4096); break;
        case 2048: GSP_S1F(2048); break;
        case 1024: GSP_S1F(1024); break;
        default: GSP_S1F(0); break;
    }
#undef GSP_S1F
    return cudaPeekAtLastError();
}

}  // namespace gsp
