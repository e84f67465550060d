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

#include <cuda_runtime.h>
#include <stdint.h>

#include "gsp_internal.h"

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

    const int s = blockIdx.y;
    const int64_t t0 = (int64_t)blockIdx.x * kFT;
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

        for (int rr0 = 2 * warp + g; rr0 < nrows; rr0 += 8 * kFU) {
            float v[kFU];
#pragma unroll
            for (int k = 0; k < kFU; ++k) {
                const int rr = rr0 + 8 * k;
                v[k] = ((unsigned)(rr - lead) < (unsigned)kFT && rbase + rr < nsamp) ? __ldg(src + (int64_t)rr * nc) : 0.f;
            }
#pragma unroll
            for (int k = 0; k < kFU; ++k) {
                const int rr = rr0 + 8 * k;
                if ((unsigned)(rr - lead) < (unsigned)kFT) dst[rr] = v[k];
            }
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

}  // namespace

bool stage1_f32_supported(const gsp_plan &p) {
    if (p.dtype != GSP_F32) return false;
    if (p.cps % kFC != 0) return false;
    const int d = p.ds;
    return d == 1 || d == 2 || d == 4 || d == 8 || d == 16 || d == 32;
}

cudaError_t launch_stage1_f32(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    const int64_t total = p.n1d * (int64_t)p.ds;
    const int64_t ntile = (total + kFT - 1) / kFT;
    if (ntile > 0x7fffffff || p.nsub > 65535) return cudaErrorInvalidValue;
    int lds = 0;
    while ((1 << lds) < p.ds) ++lds;
    dim3 grid((unsigned)ntile, (unsigned)p.nsub);
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
