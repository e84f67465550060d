// gsp_host.cu — gsp_dedisperse_host: the same two kernels fed from HOST buffers.
//
// The input is cut into time chunks of ds*Uc new rows.  Each chunk is dedispersed by a
// child plan of nsamp_c = ds*Uc + H rows (H = H1 + ds*H2, the plan's halo), which yields
// exactly Uc outputs per DM.  The H rows a chunk shares with its predecessor are copied
// device-to-device from the previous chunk's buffer (the lastdata/data carry of
// Algorithm 1), so every input byte crosses PCIe once.  H2D copies,
// kernels and D2H copies run on three streams, double buffered.

#include <cuda_runtime.h>

#include <algorithm>
#include <cstdlib>
#include <new>

#include "gsp_internal.h"

namespace gsp {

struct HostStream {
    gsp_plan *child = nullptr;   // nullptr: the parent plan is run as one chunk
    int64_t Uc = 0;              // outputs per chunk and DM
    int64_t rows_c = 0;          // input rows per chunk (ds*Uc + H)
    int64_t nchunks = 0;
    size_t elem = 1;
    void *d_in[2] = {nullptr, nullptr};
    float *d_out[2] = {nullptr, nullptr};
    cudaStream_t s_in = nullptr, s_k = nullptr, s_out = nullptr;
    cudaEvent_t e_start = nullptr;
    cudaEvent_t e_in[2] = {nullptr, nullptr}, e_k[2] = {nullptr, nullptr}, e_out[2] = {nullptr, nullptr};
};

void host_stream_destroy(HostStream *hs) {
    if (!hs) return;
    if (hs->child) gsp_plan_destroy(hs->child);
    for (int i = 0; i < 2; ++i) {
        cudaFree(hs->d_in[i]);
        cudaFree(hs->d_out[i]);
        if (hs->e_in[i]) cudaEventDestroy(hs->e_in[i]);
        if (hs->e_k[i]) cudaEventDestroy(hs->e_k[i]);
        if (hs->e_out[i]) cudaEventDestroy(hs->e_out[i]);
    }
    if (hs->e_start) cudaEventDestroy(hs->e_start);
    if (hs->s_in) cudaStreamDestroy(hs->s_in);
    if (hs->s_k) cudaStreamDestroy(hs->s_k);
    if (hs->s_out) cudaStreamDestroy(hs->s_out);
    cudaGetLastError();
    delete hs;
}

static gsp_status host_stream_create(gsp_plan *p) {
    HostStream *hs = new (std::nothrow) HostStream();
    if (!hs) return GSP_ERR_ALLOC;
    p->hs = hs;
    hs->elem = (p->dtype == GSP_U8) ? 1 : 4;
    // about 2^15 new input rows per chunk; a single chunk when the job is small
    const int64_t chunk_rows = 32768;
    int64_t Uc = std::max<int64_t>(1, chunk_rows / p->ds);
    if (p->nout <= 2 * Uc) {
        hs->child = nullptr;
        hs->Uc = p->nout;
        hs->rows_c = p->nsamp;
        hs->nchunks = 1;
    } else {
        hs->Uc = Uc;
        hs->rows_c = (int64_t)p->ds * Uc + p->halo;
        hs->nchunks = (p->nout + Uc - 1) / Uc;
        gsp_status st = gsp_plan_create(&hs->child, p->nchan, p->f_top, p->chan_bw, p->dt, hs->rows_c,
                                        p->nsub, p->subband_dm, p->dm_list.data(), p->ndm, p->ds, p->dtype);
        if (st != GSP_OK) return st;
        for (int stage = 1; stage <= 2; ++stage) {
            st = gsp_plan_set_impl(hs->child, stage, (gsp_impl)p->req_impl[stage]);
            if (st != GSP_OK) return st;
        }
        if (hs->child->nout != Uc) return GSP_ERR_CUDA;  // cannot happen: see header comment
    }
    const gsp_plan *run = hs->child ? hs->child : p;
    const int nbuf = hs->nchunks > 1 ? 2 : 1;
    cudaError_t e = cudaSuccess;
    for (int i = 0; i < nbuf && e == cudaSuccess; ++i) {
        e = cudaMalloc(&hs->d_in[i], (size_t)hs->rows_c * p->nchan * hs->elem);
        if (e == cudaSuccess) e = cudaMalloc((void **)&hs->d_out[i], (size_t)p->ndm * run->out_pitch * 4);
    }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&hs->s_in, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&hs->s_k, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&hs->s_out, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&hs->e_start, cudaEventDisableTiming);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&hs->e_in[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&hs->e_k[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&hs->e_out[i], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? GSP_ERR_ALLOC : GSP_ERR_CUDA;
    }
    return GSP_OK;
}

// out_on_device: h_out is a DEVICE array (gsp_dedisperse_host_in) — the chunk results are gathered with
// device-to-device copies and nothing but the input crosses PCIe.
gsp_status host_dedisperse(gsp_plan *p, const void *h_in, float *h_out, int64_t h_out_pitch,
                           cudaStream_t user, bool out_on_device) {
    if (!p->hs) {
        gsp_status st = host_stream_create(p);
        if (st != GSP_OK) {
            host_stream_destroy(p->hs);
            p->hs = nullptr;
            return st;
        }
    }
    HostStream *hs = p->hs;
    gsp_plan *run = hs->child ? hs->child : p;
    const size_t row_bytes = (size_t)p->nchan * hs->elem;
    const char *src = (const char *)h_in;
    const int64_t new_rows = (int64_t)p->ds * hs->Uc;

    cudaError_t e = cudaEventRecord(hs->e_start, user);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(hs->s_in, hs->e_start, 0);
    gsp_status gst = GSP_OK;

    for (int64_t k = 0; k < hs->nchunks && e == cudaSuccess && gst == GSP_OK; ++k) {
        const int b = (int)(k & 1);
        // outputs [u_lo, u_lo + Uc) of every DM; the last chunk is moved back to stay full
        const bool ragged = (k == hs->nchunks - 1) && (k * hs->Uc + hs->Uc > p->nout);
        const int64_t u_lo = ragged ? p->nout - hs->Uc : k * hs->Uc;
        const int64_t row_lo = (int64_t)p->ds * u_lo;
        // ---- input: buffer b is free once the kernels of chunk k-2 are done
        if (k >= 2) e = cudaStreamWaitEvent(hs->s_in, hs->e_k[b], 0);
        if (e != cudaSuccess) break;
        if (k == 0 || ragged) {
            e = cudaMemcpyAsync(hs->d_in[b], src + (size_t)row_lo * row_bytes,
                                (size_t)hs->rows_c * row_bytes, cudaMemcpyHostToDevice, hs->s_in);
        } else {
            // carried tail: last H rows of the previous chunk's buffer (same stream: ordered)
            const size_t tail = (size_t)p->halo * row_bytes;
            if (tail)
                e = cudaMemcpyAsync(hs->d_in[b], (const char *)hs->d_in[b ^ 1] + (size_t)new_rows * row_bytes,
                                    tail, cudaMemcpyDeviceToDevice, hs->s_in);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync((char *)hs->d_in[b] + tail,
                                    src + ((size_t)row_lo + (size_t)p->halo) * row_bytes,
                                    (size_t)new_rows * row_bytes, cudaMemcpyHostToDevice, hs->s_in);
        }
        if (e == cudaSuccess) e = cudaEventRecord(hs->e_in[b], hs->s_in);
        // ---- kernels
        if (e == cudaSuccess) e = cudaStreamWaitEvent(hs->s_k, hs->e_in[b], 0);
        if (e == cudaSuccess && k >= 2) e = cudaStreamWaitEvent(hs->s_k, hs->e_out[b], 0);
        if (e != cudaSuccess) break;
        gst = gsp_dedisperse(run, hs->d_in[b], hs->d_out[b], hs->s_k);
        if (gst != GSP_OK) break;
        e = cudaEventRecord(hs->e_k[b], hs->s_k);
        // ---- output
        if (e == cudaSuccess) e = cudaStreamWaitEvent(hs->s_out, hs->e_k[b], 0);
        if (e == cudaSuccess)
            e = cudaMemcpy2DAsync(h_out + u_lo, (size_t)h_out_pitch * 4, hs->d_out[b],
                                  (size_t)run->out_pitch * 4, (size_t)hs->Uc * 4, (size_t)p->ndm,
                                  out_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, hs->s_out);
        if (e == cudaSuccess) e = cudaEventRecord(hs->e_out[b], hs->s_out);
    }
    cudaError_t e2 = cudaStreamSynchronize(hs->s_in);
    cudaError_t e3 = cudaStreamSynchronize(hs->s_k);
    cudaError_t e4 = cudaStreamSynchronize(hs->s_out);
    if (gst != GSP_OK) return gst;
    if (e != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess || e4 != cudaSuccess) {
        cudaGetLastError();
        return GSP_ERR_CUDA;
    }
    return GSP_OK;
}

}  // namespace gsp
