// gsp_static.cu — gsp_dedisperse_static: the two-stage dedispersion for callers that must not allocate.
//
// Who this is for.  Some users of libgsp run where cudaMalloc is off limits:
//   * a real-time backend thread that is already recording data on other streams — cudaMalloc and cudaFree
//     synchronise the whole device, which stalls those streams and drops samples;
//   * a process whose device memory was carved up front by another owner (a framework's caching pool, a
//     fixed arena handed out at start-up), so that a driver allocation made behind its back either fails
//     or takes memory the owner counted on;
//   * code that runs after an "initialisation is over, nothing may allocate" point enforced by policy.
// gsp_plan_create allocates (tables, the subband workspace), so those callers cannot use plans at all.
// This entry point needs no plan: the caller passes the input, the output and the two delay tables (built
// on the host with gsp_delay_tables and copied into memory the caller already owns).  The only memory the
// method needs beyond that — the subband intermediate S' that stage 1 writes and stage 2 reads — lives in
// a fixed array inside the library image, `static_ws` below.
//
// What it costs.  The array is part of the loaded module: every GPU on which this translation unit's code
// is loaded keeps GSP_STATIC_WS_BYTES (16 MiB) of device memory until the process exits, used or not.
//
// The kernels are variants of the library's one-thread-per-output pair (Algorithm 2 of the paper applied
// twice; gsp_kernels.cu "generic"), with the same accumulation order and the same output
// scaling, so the results equal gsp_dedisperse's generic path bit for bit.  No existing code path is touched.

#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <type_traits>

#include "gsp.h"

namespace {

// The subband workspace.  In HOST code the name `static_ws` is only a handle for the runtime's symbol
// calls, not a device address; static_ws_address() below asks the runtime for the real address, once per
// device, and that address is what the kernels receive.
static __device__ __align__(256) unsigned char static_ws[GSP_STATIC_WS_BYTES];

constexpr int kMaxDevices = 64;
constexpr int kThreads = 256;
constexpr size_t kMaxTableSmem = 48 * 1024;   // the shift tables of one subband / one DM are staged in
                                              // shared memory without opting in to more than the default

std::mutex ws_mutex;
void *ws_address[kMaxDevices] = {};           // device address of static_ws on device i (0: not asked yet)

// Device address of static_ws on the CURRENT device.  The first call on a device asks the runtime
// (cudaGetSymbolAddress loads the module on that device if it is not loaded yet); later calls read the cache.
cudaError_t static_ws_address(void **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(ws_mutex);
    if (!ws_address[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, static_ws);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        ws_address[dev] = p;
    }
    *out = ws_address[dev];
    return cudaSuccess;
}

// stage 1 + downsample: one thread per S'_s[u] = sum_{k<ds} sum_{j<cps} x[u*ds + k + s1[s*cps+j]][s*cps+j]
// (un-divided), written to ws[s*n1d + u].  Every element stage 2 reads is written here first.
template <typename TIn, typename Acc>
__global__ void __launch_bounds__(kThreads)
static_stage1_kernel(const TIn *__restrict__ x, const int32_t *__restrict__ s1, Acc *__restrict__ ws,
                     int64_t n1d, int nchan, int cps, int ds) {
    extern __shared__ int32_t sh_shift[];
    const int s = blockIdx.y;
    for (int j = threadIdx.x; j < cps; j += blockDim.x) sh_shift[j] = s1[s * cps + j];
    __syncthreads();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= n1d) return;
    const TIn *col = x + (int64_t)s * cps;
    Acc tot = 0;
    for (int k = 0; k < ds; ++k) {
        const int64_t t = u * ds + k;
        for (int j = 0; j < cps; ++j) tot += (Acc)col[(t + sh_shift[j]) * (int64_t)nchan + j];
    }
    ws[(int64_t)s * n1d + u] = tot;
}

// stage 2 + store: one thread per y_d[u] = (1/ds) * sum_s S'_s[u + s2[d][s]].
// scale_mode 0: ds == 1; 1: ds a power of two (exact float multiply); 2: any ds, fl32(fl64(tot) * fl64(1/ds))
// — the same three roundings as gsp_kernels.cu; float32 input always multiplies by fl32(1/ds).
template <typename Acc>
__global__ void __launch_bounds__(kThreads)
static_stage2_kernel(const Acc *__restrict__ ws, int64_t n1d, const int32_t *__restrict__ s2,
                     float *__restrict__ out, int64_t out_pitch, int64_t nout, int nsub, int scale_mode,
                     float inv_f, double inv_d) {
    extern __shared__ int32_t sh_shift[];
    const int d = blockIdx.y;
    for (int s = threadIdx.x; s < nsub; s += blockDim.x) sh_shift[s] = s2[(int64_t)d * nsub + s];
    __syncthreads();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= nout) return;
    Acc tot = 0;
    for (int s = 0; s < nsub; ++s) tot += ws[(int64_t)s * n1d + u + sh_shift[s]];
    float y;
    if (std::is_same<Acc, float>::value) {
        y = (float)tot * inv_f;
    } else if (scale_mode == 0) {
        y = (float)tot;
    } else if (scale_mode == 1) {
        y = (float)tot * inv_f;
    } else {
        y = (float)((double)tot * inv_d);
    }
    out[(int64_t)d * out_pitch + u] = y;
}

template <typename TIn, typename Acc>
cudaError_t enqueue(const void *d_in, const int32_t *d_s1, const int32_t *d_s2, void *ws, float *d_out,
                    int64_t out_pitch, int64_t n1d, int64_t nout, int nchan, int nsub, int ndm, int ds,
                    cudaStream_t st) {
    const int cps = nchan / nsub;
    dim3 g1((unsigned)((n1d + kThreads - 1) / kThreads), (unsigned)nsub);
    static_stage1_kernel<TIn, Acc><<<g1, kThreads, (size_t)cps * sizeof(int32_t), st>>>(
        (const TIn *)d_in, d_s1, (Acc *)ws, n1d, nchan, cps, ds);
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) return e;
    const int mode = (ds == 1) ? 0 : (((ds & (ds - 1)) == 0) ? 1 : 2);
    dim3 g2((unsigned)((nout + kThreads - 1) / kThreads), (unsigned)ndm);
    static_stage2_kernel<Acc><<<g2, kThreads, (size_t)nsub * sizeof(int32_t), st>>>(
        (const Acc *)ws, n1d, d_s2, d_out, out_pitch, nout, nsub, mode, 1.0f / (float)ds, 1.0 / (double)ds);
    return cudaPeekAtLastError();
}

}  // namespace

extern "C" {

int64_t gsp_static_workspace_bytes(void) { return (int64_t)GSP_STATIC_WS_BYTES; }

gsp_status gsp_dedisperse_static(const void *d_in, gsp_dtype in_dtype, int64_t nsamp, int nchan, int nsub,
                                 int ndm, int downsamp, const int32_t *d_s1, const int32_t *d_s2,
                                 int32_t h1, int32_t h2, float *d_out, int64_t out_pitch, void *cuda_stream) {
    // ---- argument checks: host arithmetic only, before any CUDA call ----
    if (!d_in || !d_s1 || !d_s2 || !d_out) return GSP_ERR_INVALID_ARG;
    if (in_dtype != GSP_U8 && in_dtype != GSP_F32) return GSP_ERR_INVALID_ARG;
    if (nchan < 1 || nsub < 1 || nchan % nsub != 0 || ndm < 1 || downsamp < 1 || nsamp < 1) return GSP_ERR_INVALID_ARG;
    if (h1 < 0 || h2 < 0) return GSP_ERR_INVALID_ARG;
    if (nsub > 65535 || ndm > 65535) return GSP_ERR_INVALID_ARG;               // grid.y of the two launches
    if ((size_t)(nchan / nsub) * sizeof(int32_t) > kMaxTableSmem) return GSP_ERR_INVALID_ARG;
    if ((size_t)nsub * sizeof(int32_t) > kMaxTableSmem) return GSP_ERR_INVALID_ARG;
    if (in_dtype == GSP_U8 && (int64_t)nchan * 255 * downsamp > INT32_MAX) return GSP_ERR_INVALID_ARG;   // int32 sums
    const int64_t n1 = nsamp - (int64_t)h1;
    const int64_t n1d = n1 > 0 ? n1 / downsamp : 0;
    const int64_t nout = n1d - (int64_t)h2;
    if (n1 <= 0 || nout <= 0) return GSP_ERR_TOO_SHORT;
    if (out_pitch < nout) return GSP_ERR_INVALID_ARG;
    // the subband intermediate must fit the fixed array: 4 bytes per element, nsub rows of n1d
    if (n1d > (int64_t)(GSP_STATIC_WS_BYTES / 4) / nsub) return GSP_ERR_TOO_LARGE;

    // ---- the array's device address (first call on this device: one runtime query, no allocation) ----
    void *ws = nullptr;
    if (static_ws_address(&ws) != cudaSuccess) return GSP_ERR_CUDA;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e;
    if (in_dtype == GSP_U8)
        e = enqueue<uint8_t, int32_t>(d_in, d_s1, d_s2, ws, d_out, out_pitch, n1d, nout, nchan, nsub, ndm,
                                      downsamp, st);
    else
        e = enqueue<float, float>(d_in, d_s1, d_s2, ws, d_out, out_pitch, n1d, nout, nchan, nsub, ndm,
                                  downsamp, st);
    return e == cudaSuccess ? GSP_OK : GSP_ERR_CUDA;
}

}  // extern "C"
