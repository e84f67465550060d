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
//   feed      a producer warp streams 128-row x 64-byte boxes of the time-major input into a ring of
//             stages with 2-D tiled TMA loads (cp.async.bulk.tensor, SASS UTMALDG), full/empty mbarriers.
//   commit    ldmatrix.m16n16.x2.trans.b8 on the 64B-swizzled stage hands every lane ring words
//             ("one channel x 4 consecutive rows"): the byte transposition costs no ALU instruction.
//   gather    output t of channel c needs ring bytes (t + s1[c]) .. +3: lanes take consecutive
//             output words, read the two ring words that hold them (bank-conflict free for any
//             shift) and realign with PRMT.F4E; the four samples of a word are summed as
//             T += w, O += odd bytes (u16x2), E = T - (O << 8).  A warp owns 16 channels x 32 words.
//   reduce    the four 16-channel partial sums meet in shared memory, ds consecutive samples are
//             folded (shuffles up to 32, through shared memory up to 256: the DownSamp column of
//             Tables 2-3) and the result is written in the format stage 2 reads.
//
// Every input byte is fetched once (no halo re-reads between time tiles), the ring needs no
// per-channel window bookkeeping, and a 64-channel group qualifies when its largest shift fits the
// ring (max s1 <= 768 rows).  Subbands with larger shifts (low-frequency wideband data) run the LONG
// instantiation of the same kernel: a CTA owns ONE subband (CW = 16 / 32 / 64 channels) and a ring of
// up to ~200 KB (CW * ring_rows bytes, ring_rows chosen per launch from the subbands' shift spreads),
// fed by boxes of CW bytes x 8192/CW rows; what fits neither runs the wide kernel
// (gsp_stage1_wide.cu) or the windowed tile kernel (gsp_stage1.cu).

#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "gsp_internal.h"
#include "gsp_device.cuh"

namespace gsp {

namespace {

constexpr int kCG = 64;                 // channels per group (the unit of the plan's group lists)
constexpr int kRing = 1024;             // ring length in rows (= bytes per channel) of the standard instantiation
constexpr int kChunkStd = 256;          // rows per chunk of the standard instantiation (64 channels per CTA)

__device__ __forceinline__ uint32_t prmt_f4e(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("prmt.b32.f4e %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// The words of ring position 0 (tiles 0 .. NSL-1 of a committing lane) stored once more past the end of the
// ring.  Not inlined on purpose: the call is a real branch around the stores (see the call site).
struct Frag8 {
    uint32_t w[8];
};
template <int NSL>
__device__ __noinline__ void mirror_store(uint32_t *d, int P, Frag8 f) {
#pragma unroll
    for (int T = 0; T < NSL; ++T) {
        d[(16 * T) * P] = f.w[2 * T];
        d[(16 * T + 8) * P] = f.w[2 * T + 1];
    }
}

// ---------------------------------------------------------------------------------------------
// The streaming kernel.  A producer warp streams 8 KB boxes (CW bytes x 8192/CW rows) of the time-major
// input into a shared-memory ring of stages with 2-D tiled TMA loads (cp.async.bulk.tensor, SASS
// UTMALDG), guarded by full/empty mbarriers, so nstage*8 KB per CTA are in flight whatever the eight
// consumer warps are doing.  The byte transposition is done by the load itself:
// ldmatrix.m16n16.trans.b8 (new on sm_100) hands thread t of a warp the two words "channel t/4 (+8),
// rows 4(t%4)..+3" of a 16-row x 16-channel tile of the landed stage, i.e. ring words, which the
// lanes store channel-major into the ring (pitch = 4 mod 32: the 8 channels x 4 quads of a fragment
// hit 32 banks).  The boxes are written with the TMA swizzle of their row length (64 B / 32 B / none)
// so that the sixteen 16-byte rows an ldmatrix reads fall on all eight 16-byte bank groups.  Rows past
// the end of the input are zero-filled by the TMA unit (they only ever feed S-samples that are not
// emitted).
//
// Template CW = channels per CTA.  CW = 64, LONG = false is the standard instantiation: ring of 1024
// rows, two CTAs per SM, four 16-channel slices x two 128-row pieces per chunk of 256 rows.  LONG: the
// ring length is a launch argument (a multiple of the chunk), CW = channels per subband, and the eight
// warps are CW/16 slices x 128/CW row pieces (chunks of 256 / 512 / 1024 rows).
//
// SPLIT (LONG, CW = 32 / 64): every 16-channel slice streams from its OWN first row — the slice's smallest
// shift — through boxes of 16 bytes x 8192/CW rows, so the ring only has to span a slice's shift spread
// (about 16/CW of the subband's): half / a quarter of the shared memory per subband, i.e. two CTAs per SM
// where the common stream leaves room for one, and subbands that otherwise fit no ring at all.
//
// NP > 1 (gsp_dedisperse_multi, the DM ranges of a DDplan over one input): the ring is SHARED.  The
// input is fetched, transposed and committed once per chunk; every plan then gathers the chunk with
// its own stage-1 shifts (own subband DM) and folds / stores with its own downsampling and workspace.
//
// RFI (gsp_plan_set_rfi, PAPER.md:82 "RFI mitigation", :208 'mask' / 'clip'): the prologue is applied
// to the words on their way into the ring — bytes of masked channels and of clipped rows are
// replaced by the channel's pad value — so the gather never sees it and no pass over the input is added.
// ---------------------------------------------------------------------------------------------
constexpr int kStageBytes = 8192;                // one stage: a TMA box of CW bytes x 8192/CW rows (two boxes for CW = 16)
constexpr int kBoxRowsMax = 256;                 // box dimensions are limited to 256 elements
constexpr int kNStage = 5;                       // stages of the standard instantiation
constexpr int kConsumerThreads = 256;            // 8 warps; warp 8 is the producer
constexpr int kThreadsT = kConsumerThreads + 32;
constexpr int kPartBytes = 2048;                 // [slices][chunk words] uint2 = 2 KB for every CW

// shared memory: barriers | (up to 1 KB of alignment slack) | stages, 1 KB aligned for the TMA swizzle | ring | part
static constexpr size_t ring_smem(int cw, int ring_rows, int nstage) {
    return 128 + 1024 + (size_t)nstage * kStageBytes + (size_t)cw * (ring_rows + 16) + kPartBytes;
}
constexpr int kSmemStream = (int)ring_smem(kCG, kRing, kNStage);

struct RingPlanArgs {
    const int32_t *s1;     // [nchan] stage-1 shifts of this plan
    void *ws;              // subband workspace
    int64_t ws_pitch, n1d;
    int ds, lds, M, fmt;   // downsampling (power of two <= 256), its log2, plane length, WsFormat
};
struct RingArgs {
    RingPlanArgs pl[kRingMaxPlans];
    const int32_t *glist;  // groups of CW channels this launch covers
    int nglist;
    int64_t seg_rows;      // S-samples per CTA time segment (multiple of the chunk; of kRing when !LONG)
    int ring_rows, nstage; // LONG: ring length in rows (multiple of the chunk), stages in flight
    // RFI prologue (template RFI): bit t of clip_bits = input row t is clipped; per-channel mask and pad bytes
    const uint32_t *clip_bits;
    const uint8_t *chan_mask, *chan_pad;
};

template <int CW, int CPS, int NP, bool RFI, bool LONG, bool SPLIT>
__global__ void __launch_bounds__(kThreadsT, 2)
stage1_stream_u8_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ RingArgs A) {
    constexpr int NSL = CW / 16;                 // 16-channel slices of the CTA's channels
    constexpr int NPC = 8 / NSL;                 // 128-row pieces per chunk (one warp per slice and piece)
    constexpr int CH = 128 * NPC;                // rows per chunk
    constexpr int CHW = CH / 4;                  // output words per chunk
    constexpr int SR = kStageBytes / CW;         // rows per stage (TMA box); a chunk is two boxes for every CW
    constexpr int RPW = SR / 8;                  // rows of a box one warp commits
    static_assert(CH == 2 * SR && NSL * NPC == 8 && CW % CPS == 0, "geometry");
    static_assert(LONG || (CW == kCG), "the standard instantiation owns 64 channels");
    static_assert(!LONG || NP == 1, "LONG: one plan");
    static_assert(!RFI || NP == 1, "RFI prologue: one plan");
    static_assert(!SPLIT || (LONG && CW > 16), "SPLIT: per-slice streams of a long ring");

    extern __shared__ __align__(128) uint8_t smem_stream[];
    __shared__ int sh_mx;
    __shared__ int fold_scratch[8];
    const int RL = LONG ? A.ring_rows : kRing;                  // ring length in rows
    const int RW = RL >> 2;                                    // ring words per channel
    const int P = RW + 4;                                      // ring pitch in words (= 4 mod 32)
    const int nst = LONG ? A.nstage : kNStage;
    uint64_t *full = (uint64_t *)smem_stream;                  // [nst] box landed (tx bytes)
    uint64_t *empty = full + 8;                                // [nst] all consumer warps have read it
    // stages: [nst][SR rows][CW bytes] time-major, written by TMA with the swizzle of the row length (64 B:
    // 16-byte chunk index ^= (row >> 1) & 3; 32 B: ^= (row >> 2) & 1), which needs the buffer on a 1 KB boundary
    uint8_t *stage = smem_stream + 128 + ((1024u - ((smem_u32(smem_stream) + 128u) & 1023u)) & 1023u);
    uint32_t *xs = (uint32_t *)(stage + nst * kStageBytes);    // [CW][P] channel-major ring
    uint2 *part = (uint2 *)(xs + CW * P);                      // [NSL][CHW]

    const int gi = blockIdx.x % A.nglist;
    const int64_t seg = blockIdx.x / A.nglist;
    const int group = __ldg(A.glist + gi);
    const int cfirst = group * CW;
    int64_t total = 0;                                         // S-samples that feed an output (longest plan)
#pragma unroll
    for (int q = 0; q < NP; ++q) total = max(total, A.pl[q].n1d << A.pl[q].lds);
    const int64_t ta = seg * A.seg_rows;                       // ring position = (input row - ta) mod RL
    if (ta >= total) return;
    const int64_t tb = (ta + A.seg_rows < total) ? ta + A.seg_rows : total;
    const int nk = (int)((tb - ta + CH - 1) / CH);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int i = 0; i < nst; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], kConsumerThreads / 32);
        }
        sh_mx = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // chunks that must be resident before a gather: the group's largest shift over all plans
    if (threadIdx.x < CW) {
        int mx = 0;
#pragma unroll
        for (int q = 0; q < NP; ++q) mx = max(mx, __ldg(A.pl[q].s1 + cfirst + threadIdx.x));
        if (SPLIT) mx -= __ldg(A.pl[0].s1 + cfirst + (int)(threadIdx.x & ~15u));   // a slice's first channel has its smallest shift
        mx = __reduce_max_sync(CW >= 32 ? 0xffffffffu : 0x0000ffffu, mx);
        if (lane == 0) atomicMax(&sh_mx, mx);
    }
    __syncthreads();
    const int L = (sh_mx + CH - 1) / CH + 1;                   // L * CH <= RL by the host's choice of the ring
    const int nhalf = 2 * (nk + L);

    if (warp == kConsumerThreads / 32) {
        // ------------------------------------ producer ------------------------------------
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            for (int h = 0; h < nhalf; ++h) {
                while (!mbar_try_wait(&empty[st], ph ^ 1u)) __nanosleep(64);   // do not steal issue slots
                mbar_arrive_expect_tx(&full[st], kStageBytes);
                if (SPLIT) {                                   // one box of 16 bytes x SR rows per slice, from the slice's own origin
#pragma unroll
                    for (int sl = 0; sl < NSL; ++sl)
                        tma_load_2d(stage + st * kStageBytes + sl * (SR * 16), &tmap, cfirst + 16 * sl,
                                    (int)(ta + (int64_t)SR * h) + __ldg(A.pl[0].s1 + cfirst + 16 * sl), &full[st]);
                } else {
#pragma unroll
                    for (int r = 0; r < SR; r += kBoxRowsMax)  // a TMA box has at most 256 rows
                        tma_load_2d(stage + st * kStageBytes + r * CW, &tmap, cfirst, (int)(ta + (int64_t)SR * h + r),
                                    &full[st]);
                }
                if (++st == nst) {
                    st = 0;
                    ph ^= 1u;
                }
            }
        }
        return;
    }

    // ---- commit: ldmatrix.trans on bytes.  A warp owns RPW rows of the landed stage and four 16 x 16 byte tiles
    //      in it (tile T: 16-channel block T % NSL, 16-row block T / NSL); one ldmatrix.m16n16.trans.b8 hands
    //      thread t the ring words "channel t/4, rows 4(t%4)..+3" and "channel t/4 + 8, same rows" of a tile:
    //      the byte transposition costs no ALU instruction at all.  .x2: lanes 0-15 address the rows of tile 2i,
    //      lanes 16-31 those of tile 2i + 1.
    uint32_t ld_off[2];                                        // byte offset in a stage of the row this lane addresses
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int T = 2 * i + (lane >> 4);
        const int row = RPW * warp + 16 * (T / NSL) + (lane & 15);
        const uint32_t sw = (CW == 64) ? (uint32_t)((row >> 1) & 3) : (CW == 32) ? (uint32_t)((row >> 2) & 1) : 0u;
        ld_off[i] = SPLIT ? (uint32_t)((T % NSL) * (SR * 16) + row * 16)     // the slice's own box, plain rows of 16 bytes
                          : (uint32_t)(row * CW) + ((((uint32_t)(T % NSL)) ^ sw) << 4);
    }
    const int qq = (RPW / 4) * warp + (lane & 3);              // quad of a box (SR / 4 quads) this lane stores first
    uint32_t *sdst = xs + (lane >> 2) * P;
    int cst = 0;
    uint32_t cph = 0;
    int cpos = 0;                                              // ring word of the next box's first quad

    // RFI prologue state: this lane commits the 2 NSL channels 16 cb + (lane >> 2) + 8 e (cb < NSL, e < 2), index
    // k = 2 cb + e: the pad bytes of those channels, and bit k = channel k masked.  SPLIT: a slice's first row.
    uint32_t rfi_pad[2] = {0u, 0u}, rfi_cm = 0u;
    int rfi_org[NSL];
    if (RFI) {
#pragma unroll
        for (int k = 0; k < 2 * NSL; ++k) {
            const int c = cfirst + 16 * (k >> 1) + (lane >> 2) + 8 * (k & 1);
            rfi_pad[k >> 2] |= (uint32_t)__ldg(A.chan_pad + c) << (8 * (k & 3));
            if (A.chan_mask && __ldg(A.chan_mask + c)) rfi_cm |= 1u << k;
        }
#pragma unroll
        for (int cb = 0; cb < NSL; ++cb) rfi_org[cb] = SPLIT ? __ldg(A.pl[0].s1 + cfirst + 16 * cb) : 0;
    }

    // `even`: the box is the first of its chunk — only such a box can start at ring word 0 (RL is a multiple of
    // the chunk), so the odd call sites carry no mirror code at all
    auto commit = [&](int h, bool even) {
        mbar_wait(&full[cst], cph);
        const uint32_t sbase = smem_u32(stage) + (uint32_t)(cst * kStageBytes);
        uint32_t o[8];                                         // o[2T], o[2T + 1]: tile T
#pragma unroll
        for (int i = 0; i < 2; ++i)
            asm volatile("ldmatrix.sync.aligned.m16n16.x2.trans.shared.b8 {%0, %1, %2, %3}, [%4];"
                         : "=r"(o[4 * i]), "=r"(o[4 * i + 1]), "=r"(o[4 * i + 2]), "=r"(o[4 * i + 3])
                         : "r"(sbase + ld_off[i])
                         : "memory");
        // the stage is free once every lane's loads have returned
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[cst]);
        if (++cst == nst) {
            cst = 0;
            cph ^= 1u;
        }
        if (RFI) {
            // o[2T + e]: channel 16 (T % NSL) + (lane >> 2) + 8 e, input rows r0 .. r0 + 3 with
            // r0 = (the slice's first row) + SR h + 4 qq + 16 (T / NSL)
#pragma unroll
            for (int T = 0; T < 4; ++T) {
                uint32_t tm = 0u;                              // byte mask of the clipped rows of this word
                if (A.clip_bits) {
                    const int64_t r0 = ta + rfi_org[T % NSL] + (int64_t)SR * h + 4 * qq + 16 * (T / NSL);
                    const uint32_t *bw = A.clip_bits + (r0 >> 5);
                    const uint32_t sh = (uint32_t)(r0 & 31);
                    const uint32_t lo = __ldg(bw), hi = (SPLIT && sh > 28u) ? __ldg(bw + 1) : 0u;   // r0 is a multiple of 4 unless SPLIT
                    const uint32_t nib = __funnelshift_r(lo, hi, sh) & 0xfu;
                    tm = ((nib * 0x00204081u) & 0x01010101u) * 0xffu;
                }
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int k = 2 * (T % NSL) + e;
                    const uint32_t padw = __byte_perm(rfi_pad[k >> 2], 0u, 0x1111 * (k & 3));
                    const uint32_t m = tm | (uint32_t)((int32_t)(rfi_cm << (31 - k)) >> 31);
                    o[2 * T + e] = (o[2 * T + e] & ~m) | (padw & m);
                }
            }
        }
        uint32_t *d = sdst + cpos + qq;
#pragma unroll
        for (int T = 0; T < 4; ++T) {
            uint32_t *dt = d + (16 * (T % NSL)) * P + 4 * (T / NSL);
            dt[0] = o[2 * T];
            dt[8 * P] = o[2 * T + 1];
        }
        if (even && warp == 0 && cpos == 0) {                  // warp-uniform: the quad that holds ring word 0 ...
            // ... is mirrored past the end of the ring.  A real branch (a call), on purpose: with the eight mirror
            // stores if-converted into every commit (predicated off nearly always) the kernel measured 8% slower
            // and ncu counted 7.9% more shared-memory wavefronts (profiles/r2_summary.md).
            if ((lane & 3) == 0) {
                Frag8 f;
#pragma unroll
                for (int i = 0; i < 2 * NSL; ++i) f.w[i] = o[i];
                mirror_store<NSL>(d + RW, P, f);
            }
        }
        cpos += SR / 4;
        if (cpos >= RW) cpos = 0;                              // RL is a multiple of SR: a box never straddles the end
    };

    // ---- gather-side constants: warp = (16-channel slice, 128-row piece of the chunk)
    const int slice = warp % NSL, piece = warp / NSL;
    const uint32_t lane_b = 128u * piece + 4u * lane;
    uint32_t sc[NP][16];                                       // shift (+ the lane's byte offset when LONG)
#pragma unroll
    for (int q = 0; q < NP; ++q)
#pragma unroll
        for (int j = 0; j < 16; ++j)
            sc[q][j] = (uint32_t)(__ldg(A.pl[q].s1 + cfirst + 16 * slice + j) -
                                  (SPLIT ? __ldg(A.pl[q].s1 + cfirst + 16 * slice) : 0)) + (LONG ? lane_b : 0u);
    const uint8_t *cb = (const uint8_t *)(xs + (16 * slice) * P);
    const uint32_t P4 = (uint32_t)P * 4u;
    uint32_t koff = 0;                                         // (k * CH) mod RL

    // ---- reduce-side constants
    constexpr int nsb = CW / CPS, sps = CPS / 16;      // subbands per CTA, 16-channel slices per subband
    const uint16_t *part16 = (const uint16_t *)part;

    for (int h = 0; h < 2 * L; h += 2) {
        commit(h, true);
        commit(h + 1, false);
    }
    named_bar_sync(1, kConsumerThreads);

    for (int k = 0; k < nk; ++k) {
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            // --------------------------- gather chunk k with plan q's shifts ---------------------------
            // T = sum of the words mod 2^32 = E + 256*O with E / O the u16x2 sums of the even / odd
            // bytes; E < 2^32, so E = T - (O << 8) exactly and only the odd bytes need unpacking.
            uint32_t Tq[4] = {0u, 0u, 0u, 0u}, Oq[4] = {0u, 0u, 0u, 0u};   // four independent add chains
            if (LONG) {
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    uint32_t B = koff + sc[q][j];              // < 2 RL
                    B = min(B, B - (uint32_t)RL);              // mod RL (the difference wraps when B < RL)
                    const uint8_t *p = cb + j * P4 + (B & ~3u);
                    const uint32_t w = prmt_f4e(*(const uint32_t *)p, *(const uint32_t *)(p + 4), B);
                    Tq[j & 3] += w;
                    Oq[j & 3] += __byte_perm(w, 0u, 0x4341);   // bytes 1 and 3 -> u16 lanes
                }
            } else {
                const uint32_t Tb = koff + lane_b;
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const uint32_t B = Tb + sc[q][j];
                    const uint32_t Aw = B & (kRing - 4);
                    const uint8_t *p = cb + j * ((kRing / 4 + 4) * 4) + Aw;
                    const uint32_t w = prmt_f4e(*(const uint32_t *)p, *(const uint32_t *)(p + 4), B);
                    Tq[j & 3] += w;
                    Oq[j & 3] += __byte_perm(w, 0u, 0x4341);   // bytes 1 and 3 -> u16 lanes
                }
            }
            const uint32_t T = (Tq[0] + Tq[1]) + (Tq[2] + Tq[3]);
            const uint32_t O = (Oq[0] + Oq[1]) + (Oq[2] + Oq[3]);
            const uint32_t E = T - (O << 8);
            part[slice * CHW + 32 * piece + lane] =
                make_uint2(__byte_perm(E, O, 0x5410), __byte_perm(E, O, 0x7632));
            named_bar_sync(1, kConsumerThreads);               // part[] complete (last plan: chunk k's ring slot is free)

            if (q == NP - 1) {
                commit(2 * (k + L), true);
                commit(2 * (k + L) + 1, false);
                koff += CH;
                if (koff >= (uint32_t)RL) koff = 0;            // RL is a multiple of CH
            }

            // --------------------- slice reduce + downsample + store (plan q) ---------------------
            {
                const RingPlanArgs &Pq = A.pl[q];
#pragma unroll
                for (int i0 = 0; i0 < CH; i0 += kConsumerThreads) {
                    const int i = i0 + (int)threadIdx.x;
                    const int64_t t = ta + (int64_t)CH * k + i;
                    const int64_t u = t >> Pq.lds;
                    const bool mine = (i & (Pq.ds - 1)) == 0 && u < Pq.n1d;
#pragma unroll
                    for (int sb = 0; sb < nsb; ++sb) {
                        int tot = 0;
#pragma unroll
                        for (int sl = 0; sl < sps; ++sl) tot += (int)part16[(sb * sps + sl) * CH + i];
                        tot = fold_ds256(tot, Pq.ds, (int)threadIdx.x, fold_scratch, 2);
                        if (mine) {
                            const int s = group * nsb + sb;
                            if (Pq.fmt == WS_I32) {
                                ((int32_t *)Pq.ws)[(int64_t)s * Pq.ws_pitch + u] = tot;
                            } else {  // WS_PK16: W[i] = S'[i] | S'[i+M] << 16
                                uint16_t *hw = (uint16_t *)Pq.ws + 2 * ((int64_t)s * Pq.ws_pitch);
                                hw[2 * u] = (uint16_t)tot;
                                if (u >= Pq.M) hw[2 * (u - Pq.M) + 1] = (uint16_t)tot;
                            }
                        }
                    }
                }
            }
            named_bar_sync(1, kConsumerThreads);               // ring stores visible, part[] free
        }
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
static bool pow2_upto(int d, int lim) { return d >= 1 && d <= lim && (d & (d - 1)) == 0; }

bool stage1_ring_supported(const gsp_plan &p) {
    if (p.dtype != GSP_U8 || p.nsamp > 0x7fffffff) return false;
    if (p.nchan % kCG != 0) return false;
    if (!(p.cps == 16 || p.cps == 32 || p.cps == 64)) return false;
    return pow2_upto(p.ds, 256) && tma_available();
}

// Geometry of the LONG instantiation for subbands of cps channels: rows per chunk, and the ring a subband whose
// largest shift is mx needs (chunks resident before a gather, see the kernel: L = ceil(mx / chunk) + 1).
static int long_chunk(int cps) { return 128 * (8 / (cps / 16)); }
static int long_ring_rows(int cps, int mx) {
    const int ch = long_chunk(cps);
    return ch * ((mx + ch - 1) / ch + 1);
}
constexpr int kLongMinStages = 3;
// dynamic shared memory a LONG launch may ask for (the kernel also has a few static words)
static size_t long_smem_limit(const gsp_plan &p) { return p.smem_optin > 1024 ? p.smem_optin - 1024 : 0; }

// The LONG launch a subband of cps channels belongs to, and the ring it needs there: 0 = common stream, ring over
// the subband's whole shift range, two CTAs per SM; 1 = per-slice streams (SPLIT), ring over the largest shift
// spread of a 16-channel slice, two CTAs per SM; 2 = the same with one CTA per SM (cps = 16: common stream, the
// two are the same thing); -1 = fits none.
static int long_class(const gsp_plan &p, int s, int &rl) {
    const size_t half_sm = 113 * 1024;           // two CTAs per SM fit when each needs at most this
    const auto first = p.s1.begin() + (size_t)s * p.cps;
    const int mx = *std::max_element(first, first + p.cps);
    int spread = 0;
    for (int c0 = 0; c0 < p.cps; c0 += 16) {
        const auto mm = std::minmax_element(first + c0, first + c0 + 16);
        spread = std::max(spread, *mm.second - *mm.first);
    }
    rl = long_ring_rows(p.cps, mx);
    if (ring_smem(p.cps, rl, kLongMinStages + 1) <= half_sm) return 0;
    if (p.cps > 16) rl = long_ring_rows(p.cps, spread);
    if (p.cps > 16 && ring_smem(p.cps, rl, kLongMinStages + 1) <= half_sm) return 1;
    if (ring_smem(p.cps, rl, kLongMinStages) <= long_smem_limit(p)) return 2;
    return -1;
}

// Split the 64-channel groups of a plan: groups whose largest stage-1 shift fits the standard ring go to
// the streaming kernel; of the rest, groups whose subbands each fit a long ring (one CTA per subband) to
// its LONG instantiations, then the wide kernel or the windowed one.
void plan_stage1_groups(gsp_plan &p) {
    p.g_ring.clear();
    p.g_win.clear();
    for (int l = 0; l < 2; ++l) {
        p.s_wide[l].clear();
        p.ns_wide[l] = 0;
    }
    for (int l = 0; l < kLongLists; ++l) {
        p.u_long[l].clear();
        p.rl_long[l] = p.nst_long[l] = 0;
        p.seg_long[l] = p.nseg_long[l] = 0;
    }
    const int ngroups = (p.nchan + kCG - 1) / kCG;
    const bool ring = stage1_ring_supported(p);
    const bool wide = stage1_wide_supported(p);
    for (int g = 0; g < ngroups; ++g) {
        int mx = 0;
        for (int c = g * kCG; c < std::min(p.nchan, (g + 1) * kCG); ++c) mx = std::max(mx, p.s1[c]);
        if (ring && mx <= kRing - kChunkStd) {
            p.g_ring.push_back(g);
            continue;
        }
        const int s0 = g * kCG / p.cps, s1e = std::min(p.nsub, (g + 1) * kCG / p.cps);
        // long rings: every subband of the group must fit one
        bool fits_long = ring;
        int rl = 0;
        for (int s = s0; s < s1e && fits_long; ++s) fits_long = long_class(p, s, rl) >= 0;
        if (fits_long) {
            for (int s = s0; s < s1e; ++s) {
                const int l = long_class(p, s, rl);
                p.u_long[l].push_back(s);
                p.rl_long[l] = std::max(p.rl_long[l], rl);
            }
            continue;
        }
        // shifts too large for any channel-major ring: the group's subbands stream through the wide
        // kernel when every one of them fits its time-major ring, else the windowed tile kernel
        bool fits = wide && (g + 1) * kCG <= p.nchan;
        for (int s = s0; s < s1e && fits; ++s) fits = stage1_wide_slots(p, s) > 0;
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
    const int64_t want = std::max<int64_t>(1, (int64_t)p.sm_count * 3 * 6 / std::max<size_t>(1, p.g_ring.size()));
    int64_t seg = (total + want - 1) / want;
    seg = std::max<int64_t>(seg, 8 * kRing);
    seg = (seg + kRing - 1) / kRing * kRing;
    p.ring_seg_rows = seg;
    p.ring_nseg = std::max<int64_t>(1, (total + seg - 1) / seg);
    // LONG launches: stages that fit beside the ring, segments for two waves (measured: fewer, longer segments —
    // less ring warm-up per row — beat finer load balancing), long against the warm-up
    for (int l = 0; l < kLongLists; ++l) {
        if (p.u_long[l].empty()) continue;
        const size_t budget = l < 2 ? (size_t)(113 * 1024) : long_smem_limit(p);
        int nst = kLongMinStages;
        while (nst < kNStage && ring_smem(p.cps, p.rl_long[l], nst + 1) <= budget) ++nst;
        p.nst_long[l] = nst;
        const int ch = long_chunk(p.cps);
        const int64_t ctas = (int64_t)p.sm_count * (l < 2 ? 2 : 1);
        const int64_t wantl = std::max<int64_t>(1, ctas * 2 / (int64_t)p.u_long[l].size());
        int64_t sg = (total + wantl - 1) / wantl;
        sg = std::max<int64_t>(sg, 8 * (int64_t)p.rl_long[l]);
        sg = (sg + ch - 1) / ch * ch;
        p.seg_long[l] = sg;
        p.nseg_long[l] = std::max<int64_t>(1, (total + sg - 1) / sg);
    }
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn() {
    // function-local static with an initialiser: looked up once, thread-safe (C++11 magic static)
    static const EncodeTiledFn fn = []() -> EncodeTiledFn {
        void *sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        EncodeTiledFn f = nullptr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            f = (EncodeTiledFn)sym;
        cudaGetLastError();
        return f;
    }();
    return fn;
}

bool tma_available() { return encode_tiled_fn() != nullptr; }

// The input as a 2-D tensor {nchan (innermost), nsamp}, fetched in boxes of box_chan channels x box_rows rows.
// The encoded map is cached on the plan per kernel family (slot), keyed on d_in AND the box geometry, and
// re-encoded when any of them changes (L2 promotion is a function of the slot).
cudaError_t input_map(const gsp_plan &p, int slot, const void *d_in, int box_chan, int box_rows, int swizzle_bytes,
                      const CUtensorMap **tm) {
    TmapCache &c = p.tmaps[slot];
    if (c.valid && c.d_in == d_in && c.box_chan == box_chan && c.box_rows == box_rows &&
        c.swizzle_bytes == swizzle_bytes) {
        *tm = &c.tm;
        return cudaSuccess;
    }
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return cudaErrorNotSupported;
    const bool f32 = (p.dtype == GSP_F32);
    const cuuint64_t dims[2] = {(cuuint64_t)p.nchan, (cuuint64_t)p.nsamp};
    const cuuint64_t strides[1] = {(cuuint64_t)p.nchan * (f32 ? 4u : 1u)};
    const cuuint32_t box[2] = {(cuuint32_t)box_chan, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1u, 1u};
    const CUresult r = enc(&c.tm, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_UINT8, 2,
                           const_cast<void *>(d_in), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           swizzle_bytes == 64   ? CU_TENSOR_MAP_SWIZZLE_64B
                           : swizzle_bytes == 32 ? CU_TENSOR_MAP_SWIZZLE_32B
                                                 : CU_TENSOR_MAP_SWIZZLE_NONE,
                           // 16-byte rows (per-slice streams): no promotion — the neighbours of a row segment are
                           // other subbands' data, wanted thousands of rows later (measured: 2-3% faster)
                           slot == TMAP_SPLIT ? CU_TENSOR_MAP_L2_PROMOTION_NONE : CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        c.valid = false;
        return cudaErrorInvalidValue;
    }
    c.d_in = d_in;
    c.box_chan = box_chan;
    c.box_rows = box_rows;
    c.swizzle_bytes = swizzle_bytes;
    c.valid = true;
    *tm = &c.tm;
    return cudaSuccess;
}

typedef void (*Stage1StreamFn)(const CUtensorMap, const RingArgs);

template <int NP, bool RFI>
static Stage1StreamFn pick_stream(int cps) {   // channels per subband are a template parameter of the reduce step
    switch (cps) {
        case 64: return (Stage1StreamFn)stage1_stream_u8_kernel<kCG, 64, NP, RFI, false, false>;
        case 32: return (Stage1StreamFn)stage1_stream_u8_kernel<kCG, 32, NP, RFI, false, false>;
        case 16: return (Stage1StreamFn)stage1_stream_u8_kernel<kCG, 16, NP, RFI, false, false>;
        default: return nullptr;
    }
}

static Stage1StreamFn pick_stream_np(int cps, int np, bool rfi) {
    if (rfi) return np == 1 ? pick_stream<1, true>(cps) : nullptr;
    switch (np) {
        case 1: return pick_stream<1, false>(cps);
        case 2: return pick_stream<2, false>(cps);
        case 3: return pick_stream<3, false>(cps);
        case 4: return pick_stream<4, false>(cps);
        default: return nullptr;
    }
}

template <bool RFI>
static Stage1StreamFn pick_stream_long_rfi(int cps, bool split) {
    switch (cps) {
        case 64: return split ? (Stage1StreamFn)stage1_stream_u8_kernel<64, 64, 1, RFI, true, true>
                              : (Stage1StreamFn)stage1_stream_u8_kernel<64, 64, 1, RFI, true, false>;
        case 32: return split ? (Stage1StreamFn)stage1_stream_u8_kernel<32, 32, 1, RFI, true, true>
                              : (Stage1StreamFn)stage1_stream_u8_kernel<32, 32, 1, RFI, true, false>;
        case 16: return (Stage1StreamFn)stage1_stream_u8_kernel<16, 16, 1, RFI, true, false>;
        default: return nullptr;
    }
}
static Stage1StreamFn pick_stream_long(int cps, bool split, bool rfi) {   // one CTA per subband, ring length a launch argument
    return rfi ? pick_stream_long_rfi<true>(cps, split) : pick_stream_long_rfi<false>(cps, split);
}

cudaError_t configure_stage1_ring(const gsp_plan &p) {
    cudaError_t e = cudaSuccess;
    if (!p.g_ring.empty()) {
        for (int np = 1; np <= kRingMaxPlans && e == cudaSuccess; ++np)
            e = cudaFuncSetAttribute((const void *)pick_stream_np(p.cps, np, false),
                                     cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemStream);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute((const void *)pick_stream_np(p.cps, 1, true),
                                     cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemStream);
    }
    for (int split = 0; split < 2 && e == cudaSuccess; ++split) {
        if (split ? (p.u_long[1].empty() && p.u_long[2].empty()) : p.u_long[0].empty()) continue;
        for (int rfi = 0; rfi < 2 && e == cudaSuccess; ++rfi)
            e = cudaFuncSetAttribute((const void *)pick_stream_long(p.cps, split && p.cps > 16, rfi != 0),
                                     cudaFuncAttributeMaxDynamicSharedMemorySize, (int)long_smem_limit(p));
    }
    return e;
}

static RingPlanArgs ring_plan_args(const gsp_plan &q) {
    RingPlanArgs a;
    int lds = 0;
    while ((1 << lds) < q.ds) ++lds;
    a.s1 = q.d_s1;
    a.ws = q.d_ws;
    a.ws_pitch = q.ws_pitch;
    a.n1d = q.n1d;
    a.ds = q.ds;
    a.lds = lds;
    a.M = q.t2.M;
    a.fmt = (int)q.ws_format;
    return a;
}

cudaError_t launch_stage1_ring(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    if (p.g_ring.empty()) return cudaSuccess;
    const int64_t nblocks = (int64_t)p.g_ring.size() * p.ring_nseg;
    if (nblocks > 0x7fffffff) return cudaErrorInvalidValue;
    if (!(p.ws_format == WS_PK16 || p.ws_format == WS_I32)) return cudaErrorInvalidValue;
    const CUtensorMap *tm = nullptr;
    cudaError_t e = input_map(p, TMAP_RING, d_in, kCG, kStageBytes / kCG, /*swizzle_bytes=*/64, &tm);
    if (e != cudaSuccess) return e;
    RingArgs A = {};
    A.pl[0] = ring_plan_args(p);
    A.glist = p.d_g_ring;
    A.nglist = (int)p.g_ring.size();
    A.seg_rows = p.ring_seg_rows;
    A.ring_rows = kRing;
    A.nstage = kNStage;
    const bool rfi = p.rfi.enabled;
    if (rfi) {
        A.clip_bits = p.rfi.d_clip_bits;
        A.chan_mask = p.rfi.d_mask;
        A.chan_pad = p.rfi.d_pad;
    }
    Stage1StreamFn fn = pick_stream_np(p.cps, 1, rfi);
    if (!fn) return cudaErrorInvalidValue;
    fn<<<(unsigned)nblocks, kThreadsT, kSmemStream, st>>>(*tm, A);
    return cudaPeekAtLastError();
}

// The subbands whose shifts need a long ring: one CTA per subband and time segment, up to three launches
// (plan_stage1_groups: common stream / per-slice streams at two CTAs per SM, per-slice streams at one).
cudaError_t launch_stage1_ring_long(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    if (!(p.ws_format == WS_PK16 || p.ws_format == WS_I32)) return cudaErrorInvalidValue;
    cudaError_t e = cudaSuccess;
    for (int l = 0; l < kLongLists && e == cudaSuccess; ++l) {
        if (p.u_long[l].empty()) continue;
        const bool split = l > 0 && p.cps > 16;
        Stage1StreamFn fn = pick_stream_long(p.cps, split, p.rfi.enabled);
        if (!fn) return cudaErrorInvalidValue;
        const CUtensorMap *tm = nullptr;
        e = split ? input_map(p, TMAP_SPLIT, d_in, 16, kStageBytes / p.cps, /*swizzle_bytes=*/0, &tm)
                  : input_map(p, TMAP_LONG, d_in, p.cps, std::min(kStageBytes / p.cps, kBoxRowsMax),
                              /*swizzle_bytes=*/p.cps == 16 ? 0 : p.cps, &tm);
        if (e != cudaSuccess) break;
        const int64_t nblocks = (int64_t)p.u_long[l].size() * p.nseg_long[l];
        if (nblocks > 0x7fffffff) return cudaErrorInvalidValue;
        RingArgs A = {};
        A.pl[0] = ring_plan_args(p);
        A.glist = p.d_u_long[l];
        A.nglist = (int)p.u_long[l].size();
        A.seg_rows = p.seg_long[l];
        A.ring_rows = p.rl_long[l];
        A.nstage = p.nst_long[l];
        if (p.rfi.enabled) {
            A.clip_bits = p.rfi.d_clip_bits;
            A.chan_mask = p.rfi.d_mask;
            A.chan_pad = p.rfi.d_pad;
        }
        fn<<<(unsigned)nblocks, kThreadsT, ring_smem(p.cps, p.rl_long[l], p.nst_long[l]), st>>>(*tm, A);
        e = cudaPeekAtLastError();
    }
    return e;
}

// Plans that can share the ring: uint8, same input geometry, every 64-channel group of every plan streams
// through the ring kernel, no RFI prologue.
bool stage1_ring_multi_ok(gsp_plan *const *plans, int np) {
    if (np < 2 || np > kRingMaxPlans) return false;
    const gsp_plan &p0 = *plans[0];
    for (int i = 0; i < np; ++i) {
        const gsp_plan &q = *plans[i];
        if (q.dtype != GSP_U8 || q.impl[1] != GSP_IMPL_TILED || q.rfi.enabled) return false;
        if (q.nchan != p0.nchan || q.nsamp != p0.nsamp || q.nsub != p0.nsub) return false;
        if (q.g_ring.size() * (size_t)kCG != (size_t)q.nchan) return false;
        if (!(q.ws_format == WS_PK16 || q.ws_format == WS_I32)) return false;
    }
    return true;
}

cudaError_t launch_stage1_ring_multi(gsp_plan *const *plans, int np, const void *d_in, cudaStream_t st) {
    if (!stage1_ring_multi_ok(plans, np)) return cudaErrorInvalidValue;
    const gsp_plan &p0 = *plans[0];
    const CUtensorMap *tm = nullptr;
    cudaError_t e = input_map(p0, TMAP_RING, d_in, kCG, kStageBytes / kCG, /*swizzle_bytes=*/64, &tm);
    if (e != cudaSuccess) return e;
    RingArgs A = {};
    int64_t total = 0;
    for (int i = 0; i < np; ++i) {
        A.pl[i] = ring_plan_args(*plans[i]);
        total = std::max<int64_t>(total, plans[i]->n1d * (int64_t)plans[i]->ds);
    }
    A.glist = p0.d_g_ring;
    A.nglist = (int)p0.g_ring.size();
    A.seg_rows = p0.ring_seg_rows;
    A.ring_rows = kRing;
    A.nstage = kNStage;
    const int64_t nseg = (total + A.seg_rows - 1) / A.seg_rows;
    const int64_t nblocks = (int64_t)A.nglist * nseg;
    if (nblocks > 0x7fffffff) return cudaErrorInvalidValue;
    Stage1StreamFn fn = pick_stream_np(p0.cps, np, false);
    if (!fn) return cudaErrorInvalidValue;
    fn<<<(unsigned)nblocks, kThreadsT, kSmemStream, st>>>(*tm, A);
    return cudaPeekAtLastError();
}

}  // namespace gsp
