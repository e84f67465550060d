// gsp_stage1_wide.cu — streaming stage-1 kernel for uint8 subbands whose shifts fit NO channel-major
// ring of gsp_stage1_ring.cu, neither the standard 1024-row ring nor its long-ring instantiations
// (low-frequency wideband data at high subband DM: the shifts of a 16-channel slice spread over more
// than ~5,900 rows).  Since the long rings exist this kernel serves the far tail only.
//
//   S_s[t]  = sum_{c in subband s} x[t + s1[c]][c]      (Algorithm 1/2 of the paper applied per
//   S'_s[u] = sum_{k<ds} S_s[u*ds + k]   (un-divided)     subband: PAPER.md:104-166, sub-band
//                                                         method PAPER.md:100)
//
// Same scheme as the float32 streaming kernel (gsp_stage1_f32.cu), on bytes: a thread-block
// cluster owns one subband and a segment of kWSeg S-samples, CTA g of the cluster owns the
// subband's g-th 16-channel group.  The producer warp streams boxes of 256 rows x 16 channels
// (16-byte row segments, 4 KB) with 2-D tiled TMA loads into a time-major ring of NS slots; the
// ring is as long as the group's shift spread needs (up to ~200 KB = 12,800 rows).  Lanes =
// (channel, output parity): lane (c, h) reads the byte ring[t + 2j + h + s1[c]][c] for sixteen
// outputs j, and the sixteen channel lanes are summed with a transposing shuffle tree.  No
// transposition, no per-channel window bookkeeping, every input byte crosses shared memory once;
// a group's rows are read once per segment plus its shift spread.  The group sums (<= 16*255)
// stay in shared memory as u16; after a cluster barrier CTA g adds the g-th part of the segment
// over the CTAs through distributed shared memory, folds ds samples and stores S' in the format
// stage 2 reads.  Integer sums: exact in any order.

#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "gsp_internal.h"
#include "gsp_device.cuh"

namespace gsp {

namespace {

constexpr int kWC = 16;                          // channels per CTA
constexpr int kWRows = 256;                      // rows per ring slot / TMA box
constexpr int kWSlotBytes = kWRows * kWC;        // 4 KB
constexpr int kWSeg = 8192;                      // S-samples per CTA segment
constexpr int kWWarps = 8;                       // consumer warps; warp 8 is the producer
constexpr int kWThreads = (kWWarps + 1) * 32;
constexpr int kWChunk = 32 * kWWarps;            // S-samples per chunk (32 per warp) = one slot of rows
constexpr int kWMaxSlots = 52;

template <int FMT>
__global__ void __launch_bounds__(kWThreads, 2)
stage1_u8_wide_kernel(const __grid_constant__ CUtensorMap tmap, const int32_t *__restrict__ s1,
                      void *__restrict__ ws, int64_t ws_pitch, int64_t n1d, int cps, int ds, int lds, int M,
                      const int32_t *__restrict__ slist, int NS) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(128) uint8_t smem_w[];
    __shared__ int fold_scratch[8];
    uint64_t *full = (uint64_t *)smem_w;                      // [NS <= 52] box landed
    uint64_t *empty = full + kWMaxSlots;                      // [NS <= 52] all consumer warps are past the slot
    const uint8_t *ring = smem_w + 1024;                      // [NS][256 rows][16 channels]
    uint16_t *outs = (uint16_t *)(smem_w + 1024 + NS * kWSlotBytes);   // [kWSeg] this group's sums

    const int ngroups = cps / kWC;
    const int g = (int)cluster.block_rank();
    const int s = __ldg(slist + blockIdx.x / ngroups);
    const int64_t tseg = (int64_t)blockIdx.y * kWSeg;
    const int64_t total = n1d << lds;                         // tseg < total by construction of the grid
    const int segn = (int)((total - tseg < kWSeg) ? (total - tseg) : kWSeg);
    const int nk = (segn + kWChunk - 1) / kWChunk;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int c16 = lane & 15, h = lane >> 4;

    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], kWWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int c0 = s * cps + g * kWC;
    const int sh = __ldg(s1 + c0 + c16);
    int smin = sh, smax = sh;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        smin = min(smin, __shfl_xor_sync(0xffffffffu, smin, o));
        smax = max(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    }
    const int spread = smax - smin;
    const int nslot = (kWChunk * nk + spread + kWRows - 1) / kWRows;

    if (warp == kWWarps) {
        // ------------------------------------ producer ------------------------------------
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            const int64_t rbase = tseg + smin;
            for (int j = 0; j < nslot; ++j) {
                while (!mbar_try_wait(&empty[st], ph ^ 1u)) __nanosleep(64);
                mbar_arrive_expect_tx(&full[st], kWSlotBytes);
                tma_load_2d((void *)(smem_w + 1024 + st * kWSlotBytes), &tmap, c0, (int)(rbase + (int64_t)kWRows * j),
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
        const uint32_t ringb = (uint32_t)(NS * kWSlotBytes);  // ring size in bytes
        uint32_t xoff[8];                                     // ring offset of output pair (j ^ (c16 >> 1)): 4 rows per pair
#pragma unroll
        for (int j = 0; j < 8; ++j) xoff[j] = 4u * kWC * (uint32_t)(j ^ (c16 >> 1));
        uint32_t abase = (uint32_t)((32 * warp + h + (sh - smin)) * kWC + c16) % ringb;   // chunk 0
        for (int k = 0; k < nk; ++k) {
            const int r0 = kWChunk * k + 32 * warp;           // first ring row the warp touches
            // the slots this warp's rows live in — and the chunk's own slot, which it hands back below: a slot
            // is only released after its box was seen landed (see gsp_stage1_f32.cu)
            wait_upto(max((r0 + 31 + spread) >> 8, k));
            // sixteen bytes of this lane's channel (rows 2j + h), packed two per register as u16 lanes
            // register j holds the output pair (j ^ (c16 >> 1)): with this lane-dependent order the
            // transposing sum needs no selects
            uint32_t w[8];
            if (__all_sync(0xffffffffu, abase + 2u * kWC * 15u < ringb)) {   // no lane wraps in this chunk
                const uint8_t *rp = ring + abase;
#pragma unroll
                for (int j = 0; j < 8; ++j) w[j] = (uint32_t)rp[xoff[j]] | ((uint32_t)rp[xoff[j] + 2 * kWC] << 16);
            } else {
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    uint32_t a = abase + xoff[j], b = a + 2u * kWC;
                    a = (a >= ringb) ? a - ringb : a;
                    b = (b >= ringb) ? b - ringb : b;
                    w[j] = (uint32_t)ring[a] | ((uint32_t)ring[b] << 16);
                }
            }
            abase += (uint32_t)(kWChunk * kWC);
            abase = (abase >= ringb) ? abase - ringb : abase;
            // transposing sum over the 16 channel lanes on the packed pairs (sums <= 16*255 fit a u16 lane):
            // lane bits 3,2,1 select the pair, lane bit 0 the half; lane c16 ends with output j = c16
#pragma unroll
            for (int m = 4; m >= 1; m >>= 1) {
#pragma unroll
                for (int j = 0; j < m; ++j) w[j] += __shfl_xor_sync(0xffffffffu, w[j + m], 2 * m);
            }
            int v[1];
            {
                const bool up = (c16 & 1) != 0;
                const uint32_t lo = w[0] & 0xffffu, hi = w[0] >> 16;
                v[0] = (int)((up ? hi : lo) + __shfl_xor_sync(0xffffffffu, up ? lo : hi, 1));
            }
            outs[r0 + 2 * c16 + h] = (uint16_t)v[0];
            // this warp is past chunk k: it gives the chunk's slot back (one arrive per warp; the producer
            // refills the slot when all eight warps have) — no CTA barrier in the loop
            __syncwarp();
            if (lane == 0 && k < nslot) mbar_arrive(&empty[rslot]);
            if (++rslot == NS) rslot = 0;
        }
    }

    // ---- sum the groups, fold ds samples, store: CTA g takes the g-th part of the segment and reads
    //      the other CTAs' sums through distributed shared memory
    cluster_sync_publish();
    {
        const int part = kWSeg / ngroups;
        const uint16_t *src[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) src[r] = cluster.map_shared_rank(outs, r < ngroups ? r : 0);
        if (threadIdx.x < kWWarps * 32) {
            for (int i0 = g * part; i0 < (g + 1) * part; i0 += kWWarps * 32) {
                const int i = i0 + (int)threadIdx.x;
                int r = 0;
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    if (q < ngroups) r += (int)src[q][i];
                r = fold_ds256(r, ds, (int)threadIdx.x, fold_scratch, 2);
                const int64_t u = (tseg + i) >> lds;
                if ((i & (ds - 1)) == 0 && i < segn && u < n1d) {
                    if (FMT == WS_I32) {
                        ((int32_t *)ws)[(int64_t)s * ws_pitch + u] = r;
                    } else {  // WS_PK16: W[i] = S'[i] | S'[i+M] << 16
                        uint16_t *h16 = (uint16_t *)ws + 2 * ((int64_t)s * ws_pitch);
                        h16[2 * u] = (uint16_t)r;
                        if (u >= M) h16[2 * (u - M) + 1] = (uint16_t)r;
                    }
                }
            }
        }
    }
    cluster_sync_relaxed();   // remote reads are done before any CTA of the cluster exits
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
static size_t wide_smem(int ns) { return 1024 + (size_t)ns * kWSlotBytes + (size_t)kWSeg * 2; }

bool stage1_wide_supported(const gsp_plan &p) {
    if (p.dtype != GSP_U8 || p.nsamp > 0x7fffffff) return false;
    if (!(p.cps == 16 || p.cps == 32 || p.cps == 64)) return false;
    const int d = p.ds;
    if (d < 1 || d > 256 || (d & (d - 1))) return false;
    return tma_available();
}

// Ring slots subband s needs: the rows one chunk of a warp can span, the lag of the slowest warp and
// three boxes of prefetch.  0 = does not fit shared memory.
int stage1_wide_slots(const gsp_plan &p, int s) {
    int spread = 0;
    for (int c0 = s * p.cps; c0 < (s + 1) * p.cps; c0 += kWC) {
        const auto mm = std::minmax_element(p.s1.begin() + c0, p.s1.begin() + c0 + kWC);
        spread = std::max(spread, *mm.second - *mm.first);
    }
    const int ns = (kWChunk + spread + 2 * kWRows - 1) / kWRows + 1 + 3;
    return ns <= kWMaxSlots ? ns : 0;
}

// two CTAs per SM fit up to this many slots
int stage1_wide_mid_slots() { return (int)((113 * 1024 - 1024 - kWSeg * 2) / kWSlotBytes); }

typedef void (*Stage1WideFn)(const CUtensorMap, const int32_t *, void *, int64_t, int64_t, int, int, int, int,
                             const int32_t *, int);

cudaError_t configure_stage1_wide(const gsp_plan &p) {
    if (p.s_wide[0].empty() && p.s_wide[1].empty()) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute((const void *)(Stage1WideFn)stage1_u8_wide_kernel<WS_I32>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wide_smem(kWMaxSlots));
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute((const void *)(Stage1WideFn)stage1_u8_wide_kernel<WS_PK16>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wide_smem(kWMaxSlots));
    return e;
}

cudaError_t launch_stage1_wide(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    if (p.s_wide[0].empty() && p.s_wide[1].empty()) return cudaSuccess;
    if (!(p.ws_format == WS_PK16 || p.ws_format == WS_I32)) return cudaErrorInvalidValue;
    const CUtensorMap *tm = nullptr;
    cudaError_t e = input_map(p, TMAP_WIDE, d_in, kWC, kWRows, /*swizzle_bytes=*/0, &tm);
    if (e != cudaSuccess) return e;
    int lds = 0;
    while ((1 << lds) < p.ds) ++lds;
    const int64_t total = p.n1d * (int64_t)p.ds;
    const int64_t nseg = (total + kWSeg - 1) / kWSeg;
    if (nseg > 65535) return cudaErrorInvalidValue;
    const int ng = p.cps / kWC;
    Stage1WideFn fn = (p.ws_format == WS_PK16) ? (Stage1WideFn)stage1_u8_wide_kernel<WS_PK16>
                                               : (Stage1WideFn)stage1_u8_wide_kernel<WS_I32>;
    for (int l = 0; l < 2 && e == cudaSuccess; ++l) {
        if (p.s_wide[l].empty()) continue;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(p.s_wide[l].size() * ng), (unsigned)nseg);
        cfg.blockDim = dim3(kWThreads);
        cfg.dynamicSmemBytes = wide_smem(p.ns_wide[l]);
        cfg.stream = st;
        cudaLaunchAttribute attr;
        attr.id = cudaLaunchAttributeClusterDimension;
        attr.val.clusterDim.x = (unsigned)ng;
        attr.val.clusterDim.y = 1;
        attr.val.clusterDim.z = 1;
        cfg.attrs = &attr;
        cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, fn, *tm, (const int32_t *)p.d_s1, p.d_ws, p.ws_pitch, p.n1d, p.cps, p.ds, lds,
                               p.t2.M, (const int32_t *)p.d_s_wide[l], p.ns_wide[l]);
        if (e == cudaSuccess) e = cudaPeekAtLastError();
    }
    return e;
}

}  // namespace gsp
