// gsp_rfi.cu — RFI prologue of a uint8 plan: channel mask and block-wise
// zero-DM clip ("RFI mitigation" PAPER.md:82; the 'mask' and 'clip' options of prepsubband PAPER.md:208).
// The paper prints no mechanics; what is computed is readings F1-F4 of DESIGN.md §3a:
//
//   F1  x1[t][c] = mask[c] ? pad[c] : x[t][c]
//   F2  z[t] = sum_c x1[t][c]                                   (exact integer)
//   F3  per block of B rows (n rows in the ragged last one): S1 = sum z, S2 = sum z^2 (int64, exact);
//       row t is clipped iff (double)(n*z[t] - S1) > clip_sigma * sqrt((double)(n*S2 - S1*S1))
//   F4  x2[t][c] = clipped[t] ? pad[c] : x1[t][c];   dedispersion then runs on x2
//
// F1 and F4 cost no pass over the data: the stage-1 ring kernel applies them to the words on their way into
// its shared-memory ring (gsp_stage1_ring.cu, template RFI), the generic kernel at its loads.  F2/F3 need the
// whole row before any subband sum can use it, so the clip has one extra read of the input: the kernel
// below (one CTA per statistics block; byte sums with dp4a against the keep bytes 1 - mask) writes z and
// the clip bitmap the stage-1 kernels look up.

#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <vector>

#include "gsp_internal.h"

namespace gsp {

namespace {

constexpr int kZThreads = 256;

__global__ void __launch_bounds__(kZThreads)
rfi_zero_dm_kernel(const uint8_t *__restrict__ x, int64_t nsamp, int nchan, const uint8_t *__restrict__ keep,
                   int pad_sum, int B, double clip_sigma, int32_t *__restrict__ z, uint32_t *__restrict__ bits) {
    extern __shared__ int32_t zs[];                 // [B] zero-DM sums of this block's rows
    __shared__ long long red1[8], red2[8];
    __shared__ long long sh_S1;
    __shared__ double sh_rhs;
    const int64_t t0 = (int64_t)blockIdx.x * B;
    const int n = (int)((nsamp - t0 < B) ? (nsamp - t0) : B);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // ---- F1 + F2: one warp per row, two rows in flight
    const bool vec = (nchan & 15) == 0;
    for (int r = 2 * warp; r < n; r += 16) {
        unsigned acc[2] = {0u, 0u};
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            if (r + k >= n) break;
            const uint8_t *row = x + (t0 + r + k) * (int64_t)nchan;
            if (vec) {
                for (int i = lane; i < (nchan >> 4); i += 32) {
                    const uint4 v = __ldg((const uint4 *)row + i), m = __ldg((const uint4 *)keep + i);
                    acc[k] = __dp4a(v.x, m.x, acc[k]);
                    acc[k] = __dp4a(v.y, m.y, acc[k]);
                    acc[k] = __dp4a(v.z, m.z, acc[k]);
                    acc[k] = __dp4a(v.w, m.w, acc[k]);
                }
            } else {
                for (int c = lane; c < nchan; c += 32) acc[k] += (unsigned)__ldg(row + c) * (unsigned)__ldg(keep + c);
            }
        }
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const int tot = (int)__reduce_add_sync(0xffffffffu, acc[k]) + pad_sum;
            if (lane == 0 && r + k < n) {
                zs[r + k] = tot;
                z[t0 + r + k] = tot;
            }
        }
    }
    __syncthreads();

    // ---- F3: block sums (exact int64), threshold in binary64, flags -> bitmap
    long long s1 = 0, s2 = 0;
    for (int i = threadIdx.x; i < n; i += kZThreads) {
        const long long v = zs[i];
        s1 += v;
        s2 += v * v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    if (lane == 0) {
        red1[warp] = s1;
        red2[warp] = s2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long S1 = 0, S2 = 0;
        for (int w = 0; w < 8; ++w) {
            S1 += red1[w];
            S2 += red2[w];
        }
        sh_S1 = S1;
        sh_rhs = __dmul_rn(clip_sigma, sqrt((double)((long long)n * S2 - S1 * S1)));
    }
    __syncthreads();
    const long long S1 = sh_S1;
    const double rhs = sh_rhs;
    for (int i0 = 0; i0 < B; i0 += kZThreads) {                // B is a multiple of 32: words never straddle blocks
        const int i = i0 + threadIdx.x;
        const bool clip = i < n && (double)((long long)n * zs[i] - S1) > rhs;
        const unsigned m = __ballot_sync(0xffffffffu, clip);
        if (lane == 0 && i < B && t0 + i < ((nsamp + 31) & ~(int64_t)31)) bits[(t0 + i) >> 5] = m;
    }
}

}  // namespace

void rfi_free(RfiState &r) {
    cudaFree(r.d_mask);
    cudaFree(r.d_pad);
    cudaFree(r.d_keep);
    cudaFree(r.d_z);
    cudaFree(r.d_clip_bits);
    cudaFree(r.d_rest);
    r = RfiState();
}

// rows of the clip bitmap the stage-1 kernels may look up past nsamp (ring warm-up + zero-filled tail boxes)
static int64_t bitmap_words(int64_t nsamp) { return (nsamp + 32768) / 32 + 2; }

gsp_status rfi_configure(gsp_plan &p, const uint8_t *h_mask, const uint8_t *h_pad, double clip_sigma, int clip_block) {
    if (p.dtype != GSP_U8 || !h_pad) return GSP_ERR_INVALID_ARG;
    if (!(clip_sigma >= 0.0) || !(clip_sigma < 1e30)) return GSP_ERR_INVALID_ARG;
    if (clip_sigma > 0.0) {
        if (clip_block < 32 || clip_block > 8192 || clip_block % 32 != 0) return GSP_ERR_INVALID_ARG;
        if ((int64_t)clip_block * p.nchan * 255 >= ((int64_t)1 << 31)) return GSP_ERR_INVALID_ARG;   // exact int64 sums
    }
    rfi_free(p.rfi);
    RfiState &r = p.rfi;
    std::vector<uint8_t> keep((size_t)p.nchan, 1), mask((size_t)p.nchan, 0);
    r.pad_sum = 0;
    for (int c = 0; c < p.nchan; ++c)
        if (h_mask && h_mask[c]) {
            mask[c] = 1;
            keep[c] = 0;
            r.has_mask = true;
            r.pad_sum += h_pad[c];
        }
    cudaError_t e = cudaMalloc((void **)&r.d_pad, (size_t)p.nchan);
    if (e == cudaSuccess) e = cudaMemcpy(r.d_pad, h_pad, (size_t)p.nchan, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&r.d_keep, (size_t)p.nchan);
    if (e == cudaSuccess) e = cudaMemcpy(r.d_keep, keep.data(), (size_t)p.nchan, cudaMemcpyHostToDevice);
    if (e == cudaSuccess && r.has_mask) {
        e = cudaMalloc((void **)&r.d_mask, (size_t)p.nchan);
        if (e == cudaSuccess) e = cudaMemcpy(r.d_mask, mask.data(), (size_t)p.nchan, cudaMemcpyHostToDevice);
    }
    if (e == cudaSuccess && clip_sigma > 0.0) {
        e = cudaMalloc((void **)&r.d_z, (size_t)p.nsamp * sizeof(int32_t));
        if (e == cudaSuccess) e = cudaMalloc((void **)&r.d_clip_bits, (size_t)bitmap_words(p.nsamp) * 4);
        if (e == cudaSuccess) e = cudaMemset(r.d_clip_bits, 0, (size_t)bitmap_words(p.nsamp) * 4);
        if (e == cudaSuccess) e = cudaStreamSynchronize(0);
    }
    // the subbands no ring kernel takes (plan_stage1_groups: wide lists, windowed 64-channel groups)
    std::vector<int32_t> rest(p.s_wide[0]);
    rest.insert(rest.end(), p.s_wide[1].begin(), p.s_wide[1].end());
    for (int32_t g : p.g_win)
        for (int s = g * 64 / p.cps; s < std::min(p.nsub, (g + 1) * 64 / p.cps); ++s) rest.push_back(s);
    std::sort(rest.begin(), rest.end());
    r.nrest = (int)rest.size();
    if (e == cudaSuccess && r.nrest > 0) {
        e = cudaMalloc((void **)&r.d_rest, rest.size() * sizeof(int32_t));
        if (e == cudaSuccess) e = cudaMemcpy(r.d_rest, rest.data(), rest.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    }
    if (e != cudaSuccess) {
        const gsp_status st = (e == cudaErrorMemoryAllocation) ? GSP_ERR_ALLOC : GSP_ERR_CUDA;
        cudaGetLastError();
        rfi_free(p.rfi);
        return st;
    }
    r.clip_sigma = clip_sigma;
    r.clip_block = clip_sigma > 0.0 ? clip_block : 0;
    r.enabled = true;
    return GSP_OK;
}

// F2 + F3 for this call's input (no-op when the plan does not clip).
cudaError_t launch_rfi_prepass(const gsp_plan &p, const void *d_in, cudaStream_t st) {
    const RfiState &r = p.rfi;
    if (!r.enabled || !(r.clip_sigma > 0.0)) return cudaSuccess;
    const int64_t nblk = (p.nsamp + r.clip_block - 1) / r.clip_block;
    if (nblk > 0x7fffffff) return cudaErrorInvalidValue;
    rfi_zero_dm_kernel<<<(unsigned)nblk, kZThreads, (size_t)r.clip_block * 4, st>>>(
        (const uint8_t *)d_in, p.nsamp, p.nchan, r.d_keep, (int)r.pad_sum, r.clip_block, r.clip_sigma, r.d_z,
        r.d_clip_bits);
    return cudaPeekAtLastError();
}

// Diagnostics of the last call: zero-DM series and per-row clip flags (synchronises the device).
gsp_status rfi_read_back(const gsp_plan &p, int64_t *h_z, uint8_t *h_clipped) {
    const RfiState &r = p.rfi;
    if (!r.enabled || !(r.clip_sigma > 0.0)) return GSP_ERR_INVALID_ARG;
    cudaError_t e = cudaDeviceSynchronize();
    std::vector<int32_t> z((size_t)p.nsamp);
    std::vector<uint32_t> bits((size_t)bitmap_words(p.nsamp));
    if (e == cudaSuccess) e = cudaMemcpy(z.data(), r.d_z, z.size() * 4, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(bits.data(), r.d_clip_bits, bits.size() * 4, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return GSP_ERR_CUDA;
    }
    for (int64_t t = 0; t < p.nsamp; ++t) {
        if (h_z) h_z[t] = z[(size_t)t];
        if (h_clipped) h_clipped[t] = (uint8_t)((bits[(size_t)(t >> 5)] >> (t & 31)) & 1u);
    }
    return GSP_OK;
}

}  // namespace gsp
