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
// per-channel window bookkeeping, and a group qualifies when its largest shift fits the ring
// (max s1 <= 768 rows); other groups run the wide kernel (gsp_stage1_wide.cu) or the windowed
// tile kernel (gsp_stage1.cu).

#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "gsp_internal.h"
#include "gsp_device.cuh"

namespace gsp {

namespace {

constexpr int kCG = 64;                 // channels per CTA
constexpr int kRing = 1024;             // ring length in rows (= bytes per channel)
constexpr int kRW = kRing / 4;          // ring words per channel
constexpr int kChunk = 256;             // rows per chunk
constexpr int kChunkW = kChunk / 4;     // 64 quads / output words per chunk

__device__ __forceinline__ uint32_t prmt_f4e(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("prmt.b32.f4e %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// ---------------------------------------------------------------------------------------------
// The streaming kernel.  A producer warp streams 128-row x 64-byte boxes of the time-major input
// into a kNStage-deep shared-memory ring with 2-D tiled TMA loads (cp.async.bulk.tensor, SASS
// UTMALDG), guarded by full/empty mbarriers, so kNStage*8 KB per CTA are in flight whatever the eight
// consumer warps are doing.  The byte transposition is done by the load itself:
// ldmatrix.m16n16.trans.b8 (new on sm_100) hands thread t of a warp the two words "channel t/4 (+8),
// rows 4(t%4)..+3" of a 16-row x 16-channel tile of the landed stage, i.e. ring words, which the
// lanes store channel-major into the ring (pitch = 4 mod 32: the 8 channels x 4 quads of a fragment
// hit 32 banks).  The boxes are written with the TMA 64-byte swizzle so that the sixteen 16-byte rows
// an ldmatrix reads (64 bytes apart) fall on all eight 16-byte bank groups.  Rows past the end of the
// input are zero-filled by the TMA unit (they only ever feed S-samples that are not emitted).
//
// NP > 1 (gsp_dedisperse_multi, the DM ranges of a DDplan over one input): the ring is SHARED.  The
// input is fetched, transposed and committed once per chunk; every plan then gathers the chunk with
// its own stage-1 shifts (own subband DM) and folds / stores with its own downsampling and workspace.
//
// RFI (gsp_plan_set_rfi, PAPER.md:82 "RFI mitigation", :208 'mask' / 'clip'): the prologue is applied
// to the words on their way into the ring — bytes of masked channels and of clipped rows are
// replaced by the channel's pad value — so the gather never sees it and no pass over the input is added.
// ---------------------------------------------------------------------------------------------
constexpr int kHalf = 128;                       // rows per TMA stage (half a chunk)
constexpr int kStageBytes = kHalf * kCG;         // 8 KB
constexpr int kNStage = 5;
constexpr int kConsumerThreads = 256;            // 8 warps; warp 8 is the producer
constexpr int kThreadsT = kConsumerThreads + 32;
constexpr int kPitchL = kRW + 4;                 // ring pitch: = 4 mod 32, so the 32 lanes of an ldmatrix
                                                 // fragment store (8 channels x 4 quads) hit 32 banks
constexpr int kRingWordsL = kCG * kPitchL;
// barriers | (up to 1 KB of alignment slack) | stages, 1 KB aligned for the TMA swizzle | ring | part
constexpr int kSmemStream = 128 + 1024 + kNStage * kStageBytes + kRingWordsL * 4 + 4 * kChunkW * 8;

struct RingPlanArgs {
    const int32_t *s1;     // [nchan] stage-1 shifts of this plan
    void *ws;              // subband workspace
    int64_t ws_pitch, n1d;
    int ds, lds, M, fmt;   // downsampling (power of two <= 256), its log2, plane length, WsFormat
};
struct RingArgs {
    RingPlanArgs pl[kRingMaxPlans];
    const int32_t *glist;  // 64-channel groups this launch covers
    int nglist;
    int64_t seg_rows;      // S-samples per CTA time segment (multiple of kRing)
    // RFI prologue (template RFI): bit t of clip_bits = input row t is clipped; per-channel mask and pad bytes
    const uint32_t *clip_bits;
    const uint8_t *chan_mask, *chan_pad;
};

template <int CPS, int NP, bool RFI>
__global__ void __launch_bounds__(kThreadsT, 2)
stage1_stream_u8_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ RingArgs A) {
    extern __shared__ __align__(128) uint8_t smem_stream[];
    __shared__ int sh_mx;
    __shared__ int fold_scratch[8];
    uint64_t *full = (uint64_t *)smem_stream;                  // [kNStage] box landed (tx bytes)
    uint64_t *empty = full + 8;                                // [kNStage] all consumer warps have read it
    // stages: [kNStage][kHalf rows][64 B] time-major, written by TMA with the 64-byte swizzle (16-byte chunk
    // index ^= (row >> 1) & 3), which needs the buffer on a 1 KB boundary of the shared address space
    uint8_t *stage = smem_stream + 128 + ((1024u - ((smem_u32(smem_stream) + 128u) & 1023u)) & 1023u);
    uint32_t *xs = (uint32_t *)(stage + kNStage * kStageBytes);   // [kCG][kPitchL] channel-major ring
    uint2 *part = (uint2 *)(xs + kRingWordsL);                 // [4 slices][kChunkW]

    const int gi = blockIdx.x % A.nglist;
    const int64_t seg = blockIdx.x / A.nglist;
    const int group = __ldg(A.glist + gi);
    const int cfirst = group * kCG;
    int64_t total = 0;                                         // S-samples that feed an output (longest plan)
#pragma unroll
    for (int q = 0; q < NP; ++q) total = max(total, A.pl[q].n1d << A.pl[q].lds);
    const int64_t ta = seg * A.seg_rows;                       // multiple of kRing
    if (ta >= total) return;
    const int64_t tb = (ta + A.seg_rows < total) ? ta + A.seg_rows : total;
    const int nk = (int)((tb - ta + kChunk - 1) / kChunk);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int i = 0; i < kNStage; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], kConsumerThreads / 32);
        }
        sh_mx = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // chunks that must be resident before a gather: the group's largest shift over all plans
    if (threadIdx.x < kCG) {
        int mx = 0;
#pragma unroll
        for (int q = 0; q < NP; ++q) mx = max(mx, __ldg(A.pl[q].s1 + cfirst + threadIdx.x));
        mx = __reduce_max_sync(0xffffffffu, mx);
        if (lane == 0) atomicMax(&sh_mx, mx);
    }
    __syncthreads();
    const int L = (sh_mx + kChunk - 1) / kChunk + 1;
    const int nhalf = 2 * (nk + L);

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

    // RFI prologue state: this lane commits channels (lane >> 2) + 8k, k = 0..7
    uint32_t rfi_pad[2] = {0u, 0u}, rfi_cm = 0u;               // pad bytes of the 8 channels; bit k = channel k masked
    if (RFI) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int c = cfirst + (lane >> 2) + 8 * k;
            rfi_pad[k >> 2] |= (uint32_t)__ldg(A.chan_pad + c) << (8 * (k & 3));
            if (A.chan_mask && __ldg(A.chan_mask + c)) rfi_cm |= 1u << k;
        }
    }

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
        if (RFI) {
            // o[k]: channel (lane >> 2) + 8k, rows r0 .. r0 + 3 with r0 = ta + 128 h + 4 qq (a multiple of 4)
            uint32_t tm = 0u;                                  // byte mask of the clipped rows of this quad
            if (A.clip_bits) {
                const int64_t r0 = ta + (int64_t)kHalf * h + 4 * qq;
                const uint32_t nib = (__ldg(A.clip_bits + (r0 >> 5)) >> (uint32_t)(r0 & 31)) & 0xfu;
                tm = ((nib * 0x00204081u) & 0x01010101u) * 0xffu;
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const uint32_t padw = __byte_perm(rfi_pad[k >> 2], 0u, 0x1111 * (k & 3));
                const uint32_t m = tm | (uint32_t)((int32_t)(rfi_cm << (31 - k)) >> 31);
                o[k] = (o[k] & ~m) | (padw & m);
            }
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
    int sc[NP][16];
#pragma unroll
    for (int q = 0; q < NP; ++q)
#pragma unroll
        for (int j = 0; j < 16; ++j) sc[q][j] = __ldg(A.pl[q].s1 + cfirst + 16 * slice + j);
    const uint8_t *cb = (const uint8_t *)(xs + (16 * slice) * kPitchL);
    const uint32_t lane_b = 128u * half + 4u * lane;

    // ---- reduce-side constants
    constexpr int nsb = kCG / CPS, sps = CPS / 16;     // subbands per group, 16-channel slices per subband
    const uint16_t *part16 = (const uint16_t *)part;

    for (int h = 0; h < 2 * L; ++h) commit(h);
    named_bar_sync(1, kConsumerThreads);

    for (int k = 0; k < nk; ++k) {
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            // --------------------------- gather chunk k with plan q's shifts ---------------------------
            const uint32_t Tb = (((uint32_t)k * kChunk) & (kRing - 1)) + lane_b;
            // T = sum of the words mod 2^32 = E + 256*O with E / O the u16x2 sums of the even / odd
            // bytes; E < 2^32, so E = T - (O << 8) exactly and only the odd bytes need unpacking.
            uint32_t Tq[4] = {0u, 0u, 0u, 0u}, Oq[4] = {0u, 0u, 0u, 0u};   // four independent add chains
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const uint32_t B = Tb + (uint32_t)sc[q][j];
                const uint32_t Aw = B & (kRing - 4);
                const uint8_t *p = cb + j * (kPitchL * 4) + Aw;
                const uint32_t w = prmt_f4e(*(const uint32_t *)p, *(const uint32_t *)(p + 4), B);
                Tq[j & 3] += w;
                Oq[j & 3] += __byte_perm(w, 0u, 0x4341);       // bytes 1 and 3 -> u16 lanes
            }
            const uint32_t T = (Tq[0] + Tq[1]) + (Tq[2] + Tq[3]);
            const uint32_t O = (Oq[0] + Oq[1]) + (Oq[2] + Oq[3]);
            const uint32_t E = T - (O << 8);
            part[slice * kChunkW + 32 * half + lane] =
                make_uint2(__byte_perm(E, O, 0x5410), __byte_perm(E, O, 0x7632));
            named_bar_sync(1, kConsumerThreads);               // part[] complete (last plan: chunk k's ring slot is free)

            if (q == NP - 1) {
                commit(2 * (k + L));
                commit(2 * (k + L) + 1);
            }

            // --------------------- slice reduce + downsample + store (plan q) ---------------------
            {
                const RingPlanArgs &P = A.pl[q];
                const int i = threadIdx.x;
                const int64_t t = ta + (int64_t)kChunk * k + i;
                const int64_t u = t >> P.lds;
                const bool mine = (i & (P.ds - 1)) == 0 && u < P.n1d;
#pragma unroll
                for (int sb = 0; sb < nsb; ++sb) {
                    int tot = 0;
#pragma unroll
                    for (int sl = 0; sl < sps; ++sl) tot += (int)part16[(sb * sps + sl) * kChunk + i];
                    tot = fold_ds256(tot, P.ds, i, fold_scratch, 2);
                    if (mine) {
                        const int s = group * nsb + sb;
                        if (P.fmt == WS_I32) {
                            ((int32_t *)P.ws)[(int64_t)s * P.ws_pitch + u] = tot;
                        } else {  // WS_PK16: W[i] = S'[i] | S'[i+M] << 16
                            uint16_t *hw = (uint16_t *)P.ws + 2 * ((int64_t)s * P.ws_pitch);
                            hw[2 * u] = (uint16_t)tot;
                            if (u >= P.M) hw[2 * (u - P.M) + 1] = (uint16_t)tot;
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

// Split the 64-channel groups of a plan: groups whose largest stage-1 shift fits the ring go to
// the streaming kernel, the rest to the wide kernel or the windowed one.
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
            p.g_ring.push_back(g);
            continue;
        }
        // shifts too large for the channel-major ring: the group's subbands stream through the wide
        // kernel when every one of them fits its time-major ring, else the windowed tile kernel
        const int s0 = g * kCG / p.cps, s1e = std::min(p.nsub, (g + 1) * kCG / p.cps);
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

bool tma_available() { return encode_tiled_fn() != nullptr; }

// The input as a 2-D tensor {nchan (innermost), nsamp}, fetched in boxes of box_chan channels x box_rows rows.
// The encoded map is cached on the plan per kernel family (slot) and re-encoded only when d_in changes.
cudaError_t input_map(const gsp_plan &p, int slot, const void *d_in, int box_chan, int box_rows, bool swizzle64,
                      const CUtensorMap **tm) {
    TmapCache &c = p.tmaps[slot];
    if (c.d_in == d_in && c.valid) {
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
                           swizzle64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        c.valid = false;
        return cudaErrorInvalidValue;
    }
    c.d_in = d_in;
    c.valid = true;
    *tm = &c.tm;
    return cudaSuccess;
}

typedef void (*Stage1StreamFn)(const CUtensorMap, const RingArgs);

template <int NP, bool RFI>
static Stage1StreamFn pick_stream(int cps) {   // channels per subband are a template parameter of the reduce step
    switch (cps) {
        case 64: return (Stage1StreamFn)stage1_stream_u8_kernel<64, NP, RFI>;
        case 32: return (Stage1StreamFn)stage1_stream_u8_kernel<32, NP, RFI>;
        case 16: return (Stage1StreamFn)stage1_stream_u8_kernel<16, NP, RFI>;
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

cudaError_t configure_stage1_ring(const gsp_plan &p) {
    if (p.g_ring.empty()) return cudaSuccess;
    cudaError_t e = cudaSuccess;
    for (int np = 1; np <= kRingMaxPlans && e == cudaSuccess; ++np)
        e = cudaFuncSetAttribute((const void *)pick_stream_np(p.cps, np, false),
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemStream);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute((const void *)pick_stream_np(p.cps, 1, true),
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemStream);
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
    cudaError_t e = input_map(p, TMAP_RING, d_in, kCG, kHalf, /*swizzle64=*/true, &tm);
    if (e != cudaSuccess) return e;
    RingArgs A = {};
    A.pl[0] = ring_plan_args(p);
    A.glist = p.d_g_ring;
    A.nglist = (int)p.g_ring.size();
    A.seg_rows = p.ring_seg_rows;
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
    cudaError_t e = input_map(p0, TMAP_RING, d_in, kCG, kHalf, /*swizzle64=*/true, &tm);
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
    const int64_t nseg = (total + A.seg_rows - 1) / A.seg_rows;
    const int64_t nblocks = (int64_t)A.nglist * nseg;
    if (nblocks > 0x7fffffff) return cudaErrorInvalidValue;
    Stage1StreamFn fn = pick_stream_np(p0.cps, np, false);
    if (!fn) return cudaErrorInvalidValue;
    fn<<<(unsigned)nblocks, kThreadsT, kSmemStream, st>>>(*tm, A);
    return cudaPeekAtLastError();
}

}  // namespace gsp
