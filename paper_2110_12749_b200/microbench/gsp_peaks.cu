// gsp_peaks.cu — microbenchmark behind the roofline denominators of DESIGN.md §7 ("measure
// FADD vs IADD/IADD3 issue rate and the clock on the box").  Not part of libgsp; built by
// paper_2110_12749_b200/build.py (build_microbench) into paper_2110_12749_b200/gsp_peaks and run as
//     ./paper_2110_12749_b200/gsp_peaks            (prints a markdown table: profiles/r2_microbench.md)
//
// Every test runs one CTA of 1024 threads per SM (persistent, `iters` trips of an unrolled body), times the
// loop with clock64() inside the kernel and with CUDA events outside, and reports operations per clock per SM
// (max over SMs of the in-kernel cycle count) and the effective SM clock.
//
//   iadd        32-bit integer add INSTRUCTIONS (a ring of dependent adds that cannot be folded into
//               three-input IADD3s; ptxas spreads them over the ALU and FMA pipes as IADD3 / IMAD.IADD)
//   fadd        float32 adds (FADD, FMA pipe)
//   iadd+imad   adds alternating between an integer add and mad.lo.u32 x*1+acc (IMAD, FMA pipe)
//   lds32       conflict-free 32-bit shared loads at rolling offsets, one add per word (+2 ALU for the offset)
//   lds128      conflict-free 128-bit shared loads
//   k2_inner    the inner loop of stage2_tiled_kernel (packed u16 operands): per 4 shared words
//               p = (w0+w1)+(w2+w3); all += p; hi += p >> 16   -> counted as 8 operand-adds
//   k2_pk_i32   the same with int32 operands (one operand per word): 4 operand-adds per 4 words

#include <cuda_runtime.h>
#include <stdint.h>

#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>

#define CHECK(x)                                                                      \
    do {                                                                              \
        cudaError_t e_ = (x);                                                         \
        if (e_ != cudaSuccess) {                                                      \
            std::fprintf(stderr, "%s:%d %s\n", __FILE__, __LINE__, cudaGetErrorString(e_)); \
            std::exit(1);                                                             \
        }                                                                             \
    } while (0)

constexpr int kThreads = 1024;
constexpr int kAcc = 8;

template <int KIND>
__global__ void __launch_bounds__(kThreads, 1)
peak_kernel(int iters, uint32_t seed, uint32_t *sink, long long *cycles) {
    __shared__ __align__(16) uint32_t sm[8192];
    for (int i = threadIdx.x; i < 8192; i += kThreads) sm[i] = seed * (uint32_t)i + 17u;
    __syncthreads();
    uint32_t a[kAcc];
    float f[kAcc];
#pragma unroll
    for (int k = 0; k < kAcc; ++k) {
        a[k] = seed + k * threadIdx.x;
        f[k] = (float)(seed & 7) + k;
    }
    uint32_t one = (seed | 1u) / (seed | 1u);     // 1, unknown to the compiler
    if (KIND == 10 && threadIdx.x >= 512) return; // the stage-2 inner loop with 16 warps per SM, as the kernel has
    if (KIND == 11 && threadIdx.x >= 768) return; // ... and with 24
    const long long t0 = clock64();
    uint32_t off = threadIdx.x;                   // rolling, conflict-free shared offsets (steps of 33 warps' worth)
    for (int it = 0; it < iters; ++it) {
        if (KIND == 0) {
            // ring of dependent adds a[k] += a[k+1]: no two consecutive adds share a destination, so ptxas
            // cannot fold two of them into one three-input IADD3 — one instruction per add
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < kAcc; ++k) a[k] += a[(k + 1) & (kAcc - 1)];
        } else if (KIND == 1) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < kAcc; ++k) f[k] += f[(k + 1) & (kAcc - 1)];
        } else if (KIND == 2) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < kAcc; k += 2) {
                    a[k] += a[(k + 1) & (kAcc - 1)];
                    asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a[k + 1]) : "r"(a[(k + 2) & (kAcc - 1)]), "r"(one));
                }
        } else if (KIND == 3) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < kAcc; ++k) {
                    off = (off + 1056u) & 8191u;
                    a[k] += sm[off];
                }
        } else if (KIND == 4) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    off = (off + 1056u) & 2047u;
                    const uint4 w = *(const uint4 *)(sm + 4 * off);
                    a[4 * k] += w.x, a[4 * k + 1] += w.y, a[4 * k + 2] += w.z, a[4 * k + 3] += w.w;
                }
        } else if (KIND == 12) {
            // the stage-2 inner loop on 64-bit elements (four u16 planes per element): 4 LDS.64 + fold per 16 operand-adds
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < kAcc / 4; ++k) {
                    uint2 w[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        off = (off + 1056u) & 4095u;
                        w[q] = *(const uint2 *)(sm + 2 * off);
                    }
                    const uint32_t s0 = (w[0].x + w[1].x) + (w[2].x + w[3].x), s1 = (w[0].y + w[1].y) + (w[2].y + w[3].y);
                    a[4 * k] += s0;
                    a[4 * k + 1] += s0 >> 16;
                    a[4 * k + 2] += s1;
                    a[4 * k + 3] += s1 >> 16;
                }
        } else if (KIND == 7) {
            // lds128 as above plus one PREDICATED-OFF st.shared per load (the predicate is false at run time): does an
            // instruction that stores nothing still take a slot of the shared-memory pipe?
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    off = (off + 1056u) & 2047u;
                    const uint4 w = *(const uint4 *)(sm + 4 * off);
                    a[4 * k] += w.x, a[4 * k + 1] += w.y, a[4 * k + 2] += w.z, a[4 * k + 3] += w.w;
                    asm volatile("{\n.reg .pred p;\nsetp.eq.u32 p, %0, 2;\n@p st.shared.u32 [%1], %2;\n}\n" ::"r"(one),
                                 "r"((uint32_t)__cvta_generic_to_shared(sm + off)), "r"(a[k])
                                 : "memory");
                }
        } else if (KIND == 8) {
            // warp shuffles alone (one 32-bit word per lane per instruction)
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < kAcc; ++k) a[k] += __shfl_xor_sync(0xffffffffu, a[(k + 1) & (kAcc - 1)], 1 + (k & 15));
        } else if (KIND == 9) {
            // lds128 and shuffles interleaved (4 words loaded + 4 words shuffled per step): do they share a pipe?
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    off = (off + 1056u) & 2047u;
                    const uint4 w = *(const uint4 *)(sm + 4 * off);
                    a[4 * k] += w.x + __shfl_xor_sync(0xffffffffu, a[4 * k + 1], 1);
                    a[4 * k + 1] += w.y + __shfl_xor_sync(0xffffffffu, a[4 * k + 2], 2);
                    a[4 * k + 2] += w.z + __shfl_xor_sync(0xffffffffu, a[4 * k + 3], 4);
                    a[4 * k + 3] += w.w + __shfl_xor_sync(0xffffffffu, a[4 * k], 8);
                }
        } else {   // 5: packed u16 inner loop of stage 2; 6: int32 operands
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < kAcc / 2; ++k) {
                    uint32_t w[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        off = (off + 1056u) & 8191u;
                        w[q] = sm[off];
                    }
                    const uint32_t s = (w[0] + w[1]) + (w[2] + w[3]);
                    a[2 * k] += s;
                    if (KIND == 5 || KIND >= 10) a[2 * k + 1] += s >> 16;
                }
        }
    }
    const long long t1 = clock64();
    uint32_t tot = 0;
#pragma unroll
    for (int k = 0; k < kAcc; ++k) tot += a[k] + (uint32_t)f[k];
    if (tot == 0x12345678u) sink[0] = tot;         // never true in practice: keeps everything live
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

struct Result {
    const char *name, *unit;
    double per_clk_sm, total_per_s, ghz;
};

template <int KIND>
static Result run(const char *name, const char *unit, double ops_per_thread_iter, int nsm, uint32_t *sink,
                  long long *cycles) {
    const int iters = 20000;
    peak_kernel<KIND><<<nsm, kThreads>>>(200, 3u, sink, cycles);
    CHECK(cudaDeviceSynchronize());
    cudaEvent_t e0, e1;
    CHECK(cudaEventCreate(&e0));
    CHECK(cudaEventCreate(&e1));
    CHECK(cudaEventRecord(e0));
    peak_kernel<KIND><<<nsm, kThreads>>>(iters, 3u, sink, cycles);
    CHECK(cudaEventRecord(e1));
    CHECK(cudaDeviceSynchronize());
    float ms = 0.f;
    CHECK(cudaEventElapsedTime(&ms, e0, e1));
    std::vector<long long> h(nsm);
    CHECK(cudaMemcpy(h.data(), cycles, nsm * sizeof(long long), cudaMemcpyDeviceToHost));
    long long mx = 0;
    for (long long c : h) mx = c > mx ? c : mx;
    const double ops_sm = ops_per_thread_iter * kThreads * (double)iters;
    Result r;
    r.name = name;
    r.unit = unit;
    r.per_clk_sm = ops_sm / (double)mx;
    r.total_per_s = ops_sm * nsm / (ms * 1e-3);
    r.ghz = (double)mx / (ms * 1e-3) / 1e9;
    return r;
}

// `gsp_peaks pcie`: what the host link delivers for the byte pattern of one end-to-end step of config 2
// (gsp_dedisperse_host: 32 chunks of 2^15 new rows = 128 MiB contiguous host-to-device each, and per chunk a
// 2-D device-to-host copy of 1024 DM rows x 128 KiB into rows 4 MB apart), each direction alone and both at once,
// with NO kernel running: the floor of the `e2e` number.
static void pcie_probe() {
    const size_t nchan = 4096, nsamp = (size_t)1 << 20, ndm = 1024, nout = 1001282, Uc = 32768;
    const size_t in_bytes = nchan * nsamp, out_bytes = ndm * nout * 4, pitch = Uc;
    char *h_in, *d_in;
    float *h_out, *d_out;
    CHECK(cudaMallocHost(&h_in, in_bytes));
    CHECK(cudaMallocHost(&h_out, out_bytes));
    CHECK(cudaMalloc(&d_in, in_bytes));
    CHECK(cudaMalloc(&d_out, ndm * pitch * 4));
    for (size_t i = 0; i < in_bytes; i += 4096) h_in[i] = 1;
    for (size_t i = 0; i < out_bytes / 4; i += 1024) h_out[i] = 0.f;
    cudaStream_t s1, s2;
    CHECK(cudaStreamCreate(&s1));
    CHECK(cudaStreamCreate(&s2));
    const int nch = (int)((nout + Uc - 1) / Uc);
    const char *names[4] = {"host-to-device only", "device-to-host only", "both directions at once",
                            "both at once, device-to-host as ONE contiguous copy per chunk (not the output layout)"};
    std::printf("| pattern (one config-2 step: 4.29 GB in, 4.10 GB out) | time | H2D | D2H |\n|---|---|---|---|\n");
    for (int mode = 0; mode < 4; ++mode) {
        for (int rep = 0; rep < 2; ++rep) {
            CHECK(cudaDeviceSynchronize());
            cudaEvent_t e0, e1;
            CHECK(cudaEventCreate(&e0));
            CHECK(cudaEventCreate(&e1));
            CHECK(cudaEventRecord(e0, 0));
            CHECK(cudaStreamWaitEvent(s1, e0, 0));
            CHECK(cudaStreamWaitEvent(s2, e0, 0));
            for (int k = 0; k < nch; ++k) {
                size_t u = (size_t)k * Uc;
                if (u + Uc > nout) u = nout - Uc;
                if (mode != 1) CHECK(cudaMemcpyAsync(d_in + u * nchan, h_in + u * nchan, Uc * nchan, cudaMemcpyHostToDevice, s1));
                if (mode == 3)
                    CHECK(cudaMemcpyAsync(h_out + (size_t)k * Uc * ndm % (ndm * nout - Uc * ndm), d_out, Uc * 4 * ndm, cudaMemcpyDeviceToHost, s2));
                else if (mode != 0)
                    CHECK(cudaMemcpy2DAsync(h_out + u, nout * 4, d_out, pitch * 4, Uc * 4, ndm, cudaMemcpyDeviceToHost, s2));
            }
            CHECK(cudaEventRecord(e1, s1));
            CHECK(cudaStreamSynchronize(s1));
            CHECK(cudaStreamSynchronize(s2));
            CHECK(cudaDeviceSynchronize());
            float ms = 0.f;
            CHECK(cudaEventElapsedTime(&ms, e0, e1));
            (void)ms;
        }
        // wall clock over both streams (events on one stream would miss the other)
        CHECK(cudaDeviceSynchronize());
        const auto t0 = std::chrono::steady_clock::now();
        for (int k = 0; k < nch; ++k) {
            size_t u = (size_t)k * Uc;
            if (u + Uc > nout) u = nout - Uc;
            if (mode != 1) CHECK(cudaMemcpyAsync(d_in + u * nchan, h_in + u * nchan, Uc * nchan, cudaMemcpyHostToDevice, s1));
            if (mode == 3)
                CHECK(cudaMemcpyAsync(h_out + (size_t)k * Uc * ndm % (ndm * nout - Uc * ndm), d_out, Uc * 4 * ndm, cudaMemcpyDeviceToHost, s2));
            else if (mode != 0)
                CHECK(cudaMemcpy2DAsync(h_out + u, nout * 4, d_out, pitch * 4, Uc * 4, ndm, cudaMemcpyDeviceToHost, s2));
        }
        CHECK(cudaDeviceSynchronize());
        const double ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
        std::printf("| %s | %.1f ms | %.1f GB/s | %.1f GB/s |\n", names[mode], ms,
                    mode != 1 ? (double)nch * Uc * nchan / ms / 1e6 : 0.0, mode != 0 ? (double)nch * Uc * 4.0 * ndm / ms / 1e6 : 0.0);
    }
}

int main(int argc, char **argv) {
    if (argc > 1 && std::string(argv[1]) == "pcie") {
        pcie_probe();
        return 0;
    }
    cudaDeviceProp prop;
    CHECK(cudaGetDeviceProperties(&prop, 0));
    const int nsm = prop.multiProcessorCount;
    uint32_t *sink;
    long long *cycles;
    CHECK(cudaMalloc(&sink, 64));
    CHECK(cudaMalloc(&cycles, nsm * sizeof(long long)));
    std::vector<Result> res;
    res.push_back(run<0>("iadd (add.u32, ALU pipe)", "adds", 64, nsm, sink, cycles));
    res.push_back(run<1>("fadd (add.f32, FMA pipe)", "adds", 64, nsm, sink, cycles));
    res.push_back(run<2>("iadd + imad alternating (ALU + FMA pipes)", "adds", 64, nsm, sink, cycles));
    res.push_back(run<3>("lds32 (+1 add per word)", "words", 64, nsm, sink, cycles));
    res.push_back(run<4>("lds128 (+1 add per word)", "words", 64, nsm, sink, cycles));
    res.push_back(run<5>("k2_inner packed u16: 4 LDS.32 + 6 ALU per 8 operand-adds", "operand-adds", 8 * 4 * 8, nsm, sink, cycles));
    res.push_back(run<6>("k2 int32 operands: 4 LDS.32 + 4 ALU per 4 operand-adds", "operand-adds", 8 * 4 * 4, nsm, sink, cycles));
    {
        Result r = run<10>("k2_inner packed u16 with 16 warps per SM (the kernel's consumer warps)", "operand-adds", 8 * 4 * 8 / 2.0, nsm, sink, cycles);
        res.push_back(r);
        r = run<11>("k2_inner packed u16 with 24 warps per SM", "operand-adds", 8 * 4 * 8 * 0.75, nsm, sink, cycles);
        res.push_back(r);
    }
    res.push_back(run<12>("k2_inner on 64-bit elements: 4 LDS.64 + fold per 16 operand-adds", "operand-adds", 8 * 2 * 16, nsm, sink, cycles));
    res.push_back(run<7>("lds128 + one predicated-off st.shared per load (words loaded)", "words", 64, nsm, sink, cycles));
    res.push_back(run<8>("shfl (one word per lane)", "words", 64, nsm, sink, cycles));
    res.push_back(run<9>("lds128 + shfl interleaved (words loaded + words shuffled)", "words", 128, nsm, sink, cycles));
    std::printf("device: %s, %d SMs, max clock %.0f MHz\n\n", prop.name, nsm, prop.clockRate / 1e3);
    std::printf("| test | per clock per SM | whole GPU | effective SM clock |\n|---|---|---|---|\n");
    for (const Result &r : res)
        std::printf("| %s | %.1f %s | %.2f T%s/s | %.3f GHz |\n", r.name, r.per_clk_sm, r.unit, r.total_per_s / 1e12, r.unit,
                    r.ghz);
    return 0;
}
