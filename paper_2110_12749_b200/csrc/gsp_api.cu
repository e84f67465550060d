// gsp_api.cu — the C ABI of include/gsp.h: plan lifecycle, stage dispatch, getters.
// No CPU fallback exists: every compute step is a CUDA kernel of gsp_kernels.cu.

#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <new>

#include "gsp_internal.h"

using namespace gsp;

namespace {

template <typename T>
cudaError_t upload(T **dst, const std::vector<T> &src) {
    cudaError_t e = cudaMalloc((void **)dst, src.size() * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice);
}

gsp_status from_cuda(cudaError_t e) {
    if (e == cudaSuccess) return GSP_OK;
    if (e == cudaErrorMemoryAllocation) {
        cudaGetLastError();
        return GSP_ERR_ALLOC;
    }
    cudaGetLastError();
    return GSP_ERR_CUDA;
}

// Decide which kernels run and (re)allocate the workspace in the format stage 2 reads.
gsp_status resolve(gsp_plan *p) {
    int want2 = p->req_impl[2];
    if (want2 == GSP_IMPL_TILED && !p->t2.supported) return GSP_ERR_INVALID_ARG;
    const int impl2 = (want2 == GSP_IMPL_GENERIC || !p->t2.supported) ? GSP_IMPL_GENERIC : GSP_IMPL_TILED;
    int want1 = p->req_impl[1];
    const bool f32tiled = stage1_f32_supported(*p);
    const bool onestage = stage1_transpose_supported(*p);
    const bool can1 = stage1_tiled_supported(*p) || f32tiled || onestage;
    if ((want1 == GSP_IMPL_TILED || want1 == GSP_IMPL_WINDOWED) && !can1) return GSP_ERR_INVALID_ARG;
    if (want1 == GSP_IMPL_WINDOWED && (f32tiled || onestage)) return GSP_ERR_INVALID_ARG;   // uint8 subband kernel
    int impl1 = (want1 == GSP_IMPL_GENERIC || !can1) ? GSP_IMPL_GENERIC
                : (want1 == GSP_IMPL_WINDOWED ? GSP_IMPL_WINDOWED : GSP_IMPL_TILED);
    if (p->rfi.enabled) {
        // the RFI prologue lives in the ring kernel (standard and long-ring instantiations) and in the generic one:
        // the subbands of a plan that need the wide or the windowed kernel run the generic kernel (rfi.d_rest),
        // every other channel group stays on the ring kernels; a plan the ring kernels cannot take at all
        // (one-stage, fewer than 16 channels per subband, nchan not a multiple of 64) runs the generic stage 1
        const bool ring_ok = !onestage && stage1_ring_supported(*p);
        if (want1 == GSP_IMPL_WINDOWED || (want1 == GSP_IMPL_TILED && !ring_ok)) return GSP_ERR_INVALID_ARG;
        if (impl1 == GSP_IMPL_TILED && !ring_ok) impl1 = GSP_IMPL_GENERIC;
    }

    WsFormat fmt = (p->dtype == GSP_F32) ? WS_F32
                   : (impl2 == GSP_IMPL_TILED && p->t2.mode != S2_I32) ? WS_PK16 : WS_I32;
    int64_t pitch = p->n1d;
    if (impl2 == GSP_IMPL_TILED) {
        const int64_t reach = p->t2.ntile_t * p->t2.tpw * (int64_t)p->t2.M + (int64_t)p->H2 + 64;
        if (reach > pitch) pitch = reach;
    }
    pitch = (pitch + 3) / 4 * 4;
    const size_t bytes = (size_t)p->nsub * (size_t)pitch * 4;
    if (bytes != p->ws_bytes || !p->d_ws) {
        if (p->d_ws) cudaFree(p->d_ws);
        p->d_ws = nullptr;
        p->ws_bytes = 0;
        cudaError_t e = cudaMalloc(&p->d_ws, bytes);
        if (e != cudaSuccess) return from_cuda(e);
        p->ws_bytes = bytes;
    }
    // padding words are read (never stored to the output) by the tiled stage 2: keep them defined
    // (the memset runs on the legacy default stream, which non-blocking caller streams are not ordered
    // against: wait for it here, at create / set_impl time, so no later launch can race it)
    cudaError_t e = cudaMemset(p->d_ws, 0, bytes);
    if (e == cudaSuccess) e = cudaStreamSynchronize(0);
    if (e != cudaSuccess) return from_cuda(e);
    p->ws_pitch = pitch;
    p->ws_format = fmt;
    p->impl[1] = impl1;
    p->impl[2] = impl2;
    return GSP_OK;
}

}  // namespace

extern "C" {

gsp_status gsp_plan_create(gsp_plan **out_plan, int nchan, double f_top, double chan_bw, double dt,
                           int64_t nsamp, int nsub, double subband_dm, const double *dm_list,
                           int ndm, int downsamp, gsp_dtype in_dtype) {
    if (!out_plan) return GSP_ERR_INVALID_ARG;
    *out_plan = nullptr;
    gsp_status st = validate_args(nchan, f_top, chan_bw, dt, nsamp, nsub, subband_dm, dm_list, ndm,
                                  downsamp, (int)in_dtype);
    if (st != GSP_OK) return st;
    gsp_plan *p = new (std::nothrow) gsp_plan();
    if (!p) return GSP_ERR_ALLOC;
    try {
        p->nchan = nchan;
        p->nsub = nsub;
        p->ndm = ndm;
        p->ds = downsamp;
        p->f_top = f_top;
        p->chan_bw = chan_bw;
        p->dt = dt;
        p->subband_dm = subband_dm;
        p->nsamp = nsamp;
        p->dtype = in_dtype;
        p->dm_list.assign(dm_list, dm_list + ndm);
        build_delay_tables(*p);
    } catch (const std::bad_alloc &) {
        delete p;
        return GSP_ERR_ALLOC;
    }
    st = compute_extents(*p);
    if (st != GSP_OK) {
        delete p;
        return st;
    }

    cudaError_t e = cudaGetDevice(&p->device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, p->device);
    if (e != cudaSuccess) {
        delete p;
        return from_cuda(e);
    }
    p->sm_count = prop.multiProcessorCount;
    p->smem_optin = prop.sharedMemPerBlockOptin;
    const size_t smem_budget = prop.sharedMemPerBlockOptin > 4096 ? prop.sharedMemPerBlockOptin - 2048 : 0;

    try {
        plan_stage2_tiling(*p, smem_budget);
        plan_stage1_groups(*p);
        plan_stage1_f32(*p);
        p->g_all.resize((p->nchan + 63) / 64);
        for (size_t g = 0; g < p->g_all.size(); ++g) p->g_all[g] = (int32_t)g;
        e = upload(&p->d_s1, p->s1);
        if (e == cudaSuccess) e = upload(&p->d_g_all, p->g_all);
        if (e == cudaSuccess && !p->g_ring.empty()) e = upload(&p->d_g_ring, p->g_ring);
        if (e == cudaSuccess && !p->g_win.empty()) e = upload(&p->d_g_win, p->g_win);
        for (int l = 0; l < 2; ++l)
            if (e == cudaSuccess && !p->s_wide[l].empty()) e = upload(&p->d_s_wide[l], p->s_wide[l]);
        for (int l = 0; l < kLongLists; ++l)
            if (e == cudaSuccess && !p->u_long[l].empty()) e = upload(&p->d_u_long[l], p->u_long[l]);
        if (e == cudaSuccess) e = upload(&p->d_s2, p->s2);
        if (e == cudaSuccess && p->t2.supported) {
            std::vector<int4> prod;
            std::vector<int32_t> offs, rows;
            build_stage2_tables(*p, prod, offs, rows);
            e = upload(&p->d_t2_prod, prod);
            if (e == cudaSuccess) e = upload(&p->d_t2_offs, offs);
            if (e == cudaSuccess) e = upload(&p->d_t2_rows, rows);
        }
    } catch (const std::bad_alloc &) {
        gsp_plan_destroy(p);
        return GSP_ERR_ALLOC;
    }
    if (e == cudaSuccess) e = configure_kernels(*p);
    if (e == cudaSuccess) e = configure_stage1(*p);
    if (e == cudaSuccess) e = configure_stage1_ring(*p);
    if (e == cudaSuccess) e = configure_stage1_f32(*p);
    if (e == cudaSuccess) e = configure_stage1_wide(*p);
    if (e != cudaSuccess) {
        gsp_plan_destroy(p);
        return from_cuda(e);
    }
    st = resolve(p);
    if (st != GSP_OK) {
        gsp_plan_destroy(p);
        return st;
    }
    *out_plan = p;
    return GSP_OK;
}

// The plan's tables and workspace live on the device that was current at gsp_plan_create.
static bool on_plan_device(const gsp_plan *plan) {
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev == plan->device;
}

// Events of the next timed call (grows the pool on demand).
static cudaError_t next_events(gsp_plan *plan, cudaEvent_t **evs) {
    if (plan->ev_used + 3 > plan->ev.size()) {
        for (int i = 0; i < 3; ++i) {
            cudaEvent_t e;
            cudaError_t err = cudaEventCreate(&e);
            if (err != cudaSuccess) return err;
            plan->ev.push_back(e);
        }
    }
    *evs = plan->ev.data() + plan->ev_used;
    return cudaSuccess;
}

// Stage 1 of one plan (every kernel family its channel groups need).
static cudaError_t run_stage1(gsp_plan *plan, const void *d_in, cudaStream_t st) {
    cudaError_t e = launch_rfi_prepass(*plan, d_in, st);      // no-op unless the plan clips
    if (e != cudaSuccess) return e;
    if (plan->impl[1] == GSP_IMPL_TILED && plan->dtype == GSP_F32) return launch_stage1_f32(*plan, d_in, st);
    if (plan->impl[1] == GSP_IMPL_TILED && stage1_transpose_supported(*plan))
        return launch_stage1_transpose(*plan, d_in, st);   // one-stage plan: nsub == nchan
    if (plan->impl[1] == GSP_IMPL_TILED && plan->rfi.enabled) {   // prologue: ring kernels + generic for the rest
        e = launch_stage1_ring(*plan, d_in, st);
        if (e == cudaSuccess) e = launch_stage1_ring_long(*plan, d_in, st);
        if (e == cudaSuccess) e = launch_stage1_generic_list(*plan, d_in, plan->rfi.d_rest, plan->rfi.nrest, st);
        return e;
    }
    if (plan->impl[1] == GSP_IMPL_TILED) {
        e = launch_stage1_ring(*plan, d_in, st);
        if (e == cudaSuccess) e = launch_stage1_ring_long(*plan, d_in, st);
        if (e == cudaSuccess) e = launch_stage1_wide(*plan, d_in, st);
        if (e == cudaSuccess) e = launch_stage1_tiled(*plan, d_in, plan->d_g_win, (int)plan->g_win.size(), st);
        return e;
    }
    if (plan->impl[1] == GSP_IMPL_WINDOWED)
        return launch_stage1_tiled(*plan, d_in, plan->d_g_all, (int)plan->g_all.size(), st);
    return launch_stage1_generic(*plan, d_in, st);
}

static cudaError_t run_stage2(gsp_plan *plan, float *d_out, cudaStream_t st) {
    return (plan->impl[2] == GSP_IMPL_TILED) ? launch_stage2_tiled(*plan, d_out, st)
                                             : launch_stage2_generic(*plan, d_out, st);
}

gsp_status gsp_dedisperse(gsp_plan *plan, const void *d_in, float *d_out, void *cuda_stream) {
    if (!plan || !d_in || !d_out) return GSP_ERR_INVALID_ARG;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return GSP_ERR_INVALID_ARG;
    if (!on_plan_device(plan)) return GSP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaSuccess;
    cudaEvent_t *evs = nullptr;
    if (plan->timing) {
        e = next_events(plan, &evs);
        if (e == cudaSuccess) e = cudaEventRecord(evs[0], st);
    }
    if (e == cudaSuccess) e = run_stage1(plan, d_in, st);
    if (e == cudaSuccess && evs) e = cudaEventRecord(evs[1], st);
    if (e == cudaSuccess) e = run_stage2(plan, d_out, st);
    if (e == cudaSuccess && evs) {
        e = cudaEventRecord(evs[2], st);
        if (e == cudaSuccess) plan->ev_used += 3;
    }
    return from_cuda(e);
}

// The longest run of plans (up to 4) starting at plans[0] that can share one stage-1 launch: kind 1 = float32
// streaming kernel, 2 = uint8 ring, 0 = none (the plan runs its own stage 1).
static int multi_group(gsp_plan *const *plans, int avail, int *kind) {
    *kind = 0;
    for (int m = std::min(avail, 4); m >= 2; --m) {
        bool f32ok = stage1_f32_multi_ok(plans, m);
        for (int j = 0; j < m && f32ok; ++j) f32ok = plans[j]->dtype == GSP_F32 && plans[j]->impl[1] == GSP_IMPL_TILED;
        if (f32ok) {
            *kind = 1;
            return m;
        }
        if (stage1_ring_multi_ok(plans, m)) {
            *kind = 2;
            return m;
        }
    }
    return 1;
}

static int stage1_launches(const gsp_plan *plan) { return gsp_plan_launches_per_call(plan) - 1; }

gsp_status gsp_plan_reserve_multi(gsp_plan *plan) {
    if (!plan || !on_plan_device(plan)) return GSP_ERR_INVALID_ARG;
    return from_cuda(reserve_stage1_f32_shared(*plan));
}

int32_t gsp_dedisperse_multi_launches(gsp_plan *const *plans, int nplans) {
    if (!plans || nplans < 1) return 0;
    int n_launch = nplans;                                     // stage 2: one kernel per plan
    for (int i = 0; i < nplans;) {
        if (!plans[i]) return 0;
        int kind = 0;
        const int n = multi_group(plans + i, nplans - i, &kind);
        n_launch += kind == 1 ? stage1_f32_multi_launches(plans + i, n) : kind == 2 ? 1 : stage1_launches(plans[i]);
        i += n;
    }
    return n_launch;
}

gsp_status gsp_dedisperse_multi(gsp_plan *const *plans, int nplans, const void *d_in, float *const *d_outs,
                                void *cuda_stream) {
    if (!plans || !d_outs || !d_in || nplans < 1) return GSP_ERR_INVALID_ARG;
    for (int i = 0; i < nplans; ++i) {
        if (!plans[i] || !d_outs[i] || ((uintptr_t)d_outs[i] & 15)) return GSP_ERR_INVALID_ARG;
        if (!on_plan_device(plans[i])) return GSP_ERR_INVALID_ARG;
        for (int j = 0; j < i; ++j)
            if (plans[j] == plans[i]) return GSP_ERR_INVALID_ARG;   // shared workspace
    }
    if ((uintptr_t)d_in & 15) return GSP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    gsp_plan *lead = plans[0];
    cudaError_t e = cudaSuccess;
    cudaEvent_t *evs = nullptr;
    if (lead->timing) {
        e = next_events(lead, &evs);
        if (e == cudaSuccess) e = cudaEventRecord(evs[0], st);
    }
    // stage 1 of every plan first (each plan owns its workspace), consecutive plans sharing one launch where
    // they can: float32 plans and uint8 plans each on ONE shared ring (input fetched once, a gather per plan)
    for (int i = 0; i < nplans && e == cudaSuccess;) {
        int kind = 0;
        const int n = multi_group(plans + i, nplans - i, &kind);
        if (kind == 1) e = launch_stage1_f32_multi(plans + i, n, d_in, st);
        else if (kind == 2) e = launch_stage1_ring_multi(plans + i, n, d_in, st);
        else e = run_stage1(plans[i], d_in, st);
        i += n;
    }
    if (e == cudaSuccess && evs) e = cudaEventRecord(evs[1], st);
    for (int i = 0; i < nplans && e == cudaSuccess; ++i) e = run_stage2(plans[i], d_outs[i], st);
    if (e == cudaSuccess && evs) {
        e = cudaEventRecord(evs[2], st);
        if (e == cudaSuccess) lead->ev_used += 3;
    }
    return from_cuda(e);
}

gsp_status gsp_dedisperse_host(gsp_plan *plan, const void *h_in, float *h_out, int64_t h_out_pitch,
                               void *cuda_stream) {
    if (!plan || !h_in || !h_out || h_out_pitch < plan->nout) return GSP_ERR_INVALID_ARG;
    if (!on_plan_device(plan)) return GSP_ERR_INVALID_ARG;
    if (plan->rfi.enabled) return GSP_ERR_INVALID_ARG;   // clip blocks are defined on the whole input, not on chunks
    return host_dedisperse(plan, h_in, h_out, h_out_pitch, (cudaStream_t)cuda_stream);
}

gsp_status gsp_dedisperse_host_in(gsp_plan *plan, const void *h_in, float *d_out, int64_t d_out_pitch,
                                  void *cuda_stream) {
    if (!plan || !h_in || !d_out || d_out_pitch < plan->nout) return GSP_ERR_INVALID_ARG;
    if (!on_plan_device(plan)) return GSP_ERR_INVALID_ARG;
    if (plan->rfi.enabled) return GSP_ERR_INVALID_ARG;   // as gsp_dedisperse_host
    return host_dedisperse(plan, h_in, d_out, d_out_pitch, (cudaStream_t)cuda_stream, /*out_on_device=*/true);
}

gsp_status gsp_plan_destroy(gsp_plan *plan) {
    if (!plan) return GSP_OK;
    if (plan->hs) host_stream_destroy(plan->hs);
    cudaFree(plan->d_s1);
    cudaFree(plan->d_s2);
    cudaFree(plan->d_g_ring);
    cudaFree(plan->d_g_win);
    cudaFree(plan->d_s_wide[0]);
    cudaFree(plan->d_s_wide[1]);
    for (int l = 0; l < kLongLists; ++l) cudaFree(plan->d_u_long[l]);
    cudaFree(plan->d_g_all);
    cudaFree(plan->d_ws);
    cudaFree(plan->d_f32_part);
    cudaFree(plan->d_t2_prod);
    cudaFree(plan->d_t2_offs);
    cudaFree(plan->d_t2_rows);
    rfi_free(plan->rfi);
    for (auto &ev : plan->ev) cudaEventDestroy(ev);
    cudaGetLastError();
    delete plan;
    return GSP_OK;
}

int64_t gsp_plan_nout(const gsp_plan *p) { return p ? p->nout : 0; }
int64_t gsp_plan_out_pitch(const gsp_plan *p) { return p ? p->out_pitch : 0; }
int64_t gsp_plan_halo(const gsp_plan *p) { return p ? p->halo : 0; }
int64_t gsp_plan_n1(const gsp_plan *p) { return p ? p->n1 : 0; }
int64_t gsp_plan_n1d(const gsp_plan *p) { return p ? p->n1d : 0; }
int32_t gsp_plan_h1(const gsp_plan *p) { return p ? p->H1 : 0; }
int32_t gsp_plan_h2(const gsp_plan *p) { return p ? p->H2 : 0; }
int32_t gsp_plan_ndm(const gsp_plan *p) { return p ? p->ndm : 0; }
const int32_t *gsp_plan_stage1_shifts(const gsp_plan *p) { return p ? p->s1.data() : nullptr; }
const int32_t *gsp_plan_stage2_shifts(const gsp_plan *p) { return p ? p->s2.data() : nullptr; }
int64_t gsp_plan_workspace_bytes(const gsp_plan *p) { return p ? (int64_t)p->ws_bytes : 0; }

gsp_status gsp_plan_set_impl(gsp_plan *plan, int stage, gsp_impl impl) {
    if (!plan || (stage != 1 && stage != 2)) return GSP_ERR_INVALID_ARG;
    if (impl != GSP_IMPL_AUTO && impl != GSP_IMPL_GENERIC && impl != GSP_IMPL_TILED &&
        !(impl == GSP_IMPL_WINDOWED && stage == 1))
        return GSP_ERR_INVALID_ARG;
    if (plan->hs) {  // the host-buffer path caches a child plan with the old selection
        host_stream_destroy(plan->hs);
        plan->hs = nullptr;
    }
    const int old = plan->req_impl[stage];
    plan->req_impl[stage] = impl;
    gsp_status st = resolve(plan);
    if (st != GSP_OK) {
        plan->req_impl[stage] = old;
        resolve(plan);
    }
    return st;
}

gsp_status gsp_plan_set_rfi(gsp_plan *plan, const uint8_t *h_chan_mask, const uint8_t *h_chan_pad, double clip_sigma,
                            int32_t clip_block) {
    if (!plan || !on_plan_device(plan)) return GSP_ERR_INVALID_ARG;
    if (plan->hs) {
        host_stream_destroy(plan->hs);
        plan->hs = nullptr;
    }
    if (!h_chan_pad) {   // clear
        rfi_free(plan->rfi);
        return resolve(plan);
    }
    gsp_status st = rfi_configure(*plan, h_chan_mask, h_chan_pad, clip_sigma, clip_block);
    if (st != GSP_OK) return st;
    st = resolve(plan);
    if (st != GSP_OK) {   // e.g. a forced kernel that has no prologue: undo
        rfi_free(plan->rfi);
        resolve(plan);
    }
    return st;
}

gsp_status gsp_plan_rfi_last(const gsp_plan *plan, int64_t *h_zero_dm, uint8_t *h_clipped) {
    if (!plan || !on_plan_device(plan)) return GSP_ERR_INVALID_ARG;
    return rfi_read_back(*plan, h_zero_dm, h_clipped);
}

int32_t gsp_plan_get_impl(const gsp_plan *plan, int stage) {
    if (!plan || (stage != 1 && stage != 2)) return -1;
    return plan->impl[stage];
}

int32_t gsp_plan_launches_per_call(const gsp_plan *plan) {
    if (!plan) return 0;
    int n = 2;  // one kernel per stage ...
    if (plan->impl[1] == GSP_IMPL_TILED && plan->dtype == GSP_U8 && !stage1_transpose_supported(*plan)) {
        // ... or one stage-1 launch per kernel that has channel groups: ring, long rings and wide (two lists
        // each), windowed
        n = 1 + (plan->g_ring.empty() ? 0 : 1) + (plan->s_wide[0].empty() ? 0 : 1) +
            (plan->s_wide[1].empty() ? 0 : 1) + (plan->u_long[0].empty() ? 0 : 1) +
            (plan->u_long[1].empty() ? 0 : 1) + (plan->u_long[2].empty() ? 0 : 1) + (plan->g_win.empty() ? 0 : 1);
        if (plan->rfi.enabled)   // wide and windowed subbands share ONE launch of the generic kernel
            n = 1 + (plan->g_ring.empty() ? 0 : 1) + (plan->u_long[0].empty() ? 0 : 1) +
                (plan->u_long[1].empty() ? 0 : 1) + (plan->u_long[2].empty() ? 0 : 1) + (plan->rfi.nrest > 0 ? 1 : 0);
    }
    if (plan->rfi.enabled && plan->rfi.clip_sigma > 0.0) ++n;   // zero-DM statistics pass of the clip
    return n;
}

gsp_status gsp_plan_stage1_split_n(const gsp_plan *plan, int32_t *counts, int32_t ncounts, int32_t *navailable) {
    if (navailable) *navailable = GSP_STAGE1_SPLIT_COUNTS;
    if (!plan || !counts || ncounts < 0) return GSP_ERR_INVALID_ARG;
    int32_t all[GSP_STAGE1_SPLIT_COUNTS];
    all[0] = (int32_t)plan->g_ring.size();
    all[1] = (int32_t)plan->s_wide[0].size();
    all[2] = (int32_t)plan->s_wide[1].size();
    all[3] = (int32_t)plan->g_win.size();
    all[4] = stage1_f32_streams(*plan) ? 1 : 0;
    all[5] = (int32_t)(plan->u_long[0].size() + plan->u_long[1].size());
    all[6] = (int32_t)plan->u_long[2].size();
    if (plan->dtype != GSP_U8)   // uint8 kernels
        all[0] = all[1] = all[2] = all[3] = all[5] = all[6] = 0;
    for (int i = 0; i < ncounts && i < GSP_STAGE1_SPLIT_COUNTS; ++i) counts[i] = all[i];
    return GSP_OK;
}

gsp_status gsp_plan_stage1_split(const gsp_plan *plan, int32_t counts[7]) {
    return gsp_plan_stage1_split_n(plan, counts, 7, nullptr);
}

gsp_status gsp_plan_enable_stage_timing(gsp_plan *plan, int enable) {
    if (!plan) return GSP_ERR_INVALID_ARG;
    plan->timing = enable != 0;
    plan->ev_used = 0;
    return GSP_OK;
}

gsp_status gsp_plan_last_stage_ms(gsp_plan *plan, float *ms1, float *ms2) {
    if (!plan || !ms1 || !ms2 || !plan->timing || plan->ev_used < 3) return GSP_ERR_INVALID_ARG;
    cudaEvent_t *evs = plan->ev.data() + plan->ev_used - 3;
    cudaError_t e = cudaEventSynchronize(evs[2]);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms1, evs[0], evs[1]);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms2, evs[1], evs[2]);
    return from_cuda(e);
}

gsp_status gsp_plan_stage_ms_total(gsp_plan *plan, double *ms1, double *ms2, int32_t *ncalls) {
    if (!plan || !ms1 || !ms2 || !ncalls || !plan->timing) return GSP_ERR_INVALID_ARG;
    *ms1 = *ms2 = 0.0;
    *ncalls = (int32_t)(plan->ev_used / 3);
    if (plan->ev_used == 0) return GSP_OK;
    cudaError_t e = cudaEventSynchronize(plan->ev[plan->ev_used - 1]);
    for (size_t i = 0; i < plan->ev_used && e == cudaSuccess; i += 3) {
        float a = 0.f, b = 0.f;
        e = cudaEventElapsedTime(&a, plan->ev[i], plan->ev[i + 1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&b, plan->ev[i + 1], plan->ev[i + 2]);
        *ms1 += a;
        *ms2 += b;
    }
    return from_cuda(e);
}

gsp_status gsp_delay_tables(int nchan, double f_top, double chan_bw, double dt, int nsub,
                            double subband_dm, const double *dm_list, int ndm, int downsamp,
                            int32_t *s1, int32_t *s2) {
    if (!s1 || !s2) return GSP_ERR_INVALID_ARG;
    gsp_status st = validate_args(nchan, f_top, chan_bw, dt, 1, nsub, subband_dm, dm_list, ndm,
                                  downsamp, GSP_U8);
    if (st != GSP_OK) return st;
    try {
        gsp_plan p;
        p.nchan = nchan;
        p.nsub = nsub;
        p.ndm = ndm;
        p.ds = downsamp;
        p.f_top = f_top;
        p.chan_bw = chan_bw;
        p.dt = dt;
        p.subband_dm = subband_dm;
        p.dm_list.assign(dm_list, dm_list + ndm);
        build_delay_tables(p);
        std::memcpy(s1, p.s1.data(), p.s1.size() * sizeof(int32_t));
        std::memcpy(s2, p.s2.data(), p.s2.size() * sizeof(int32_t));
    } catch (const std::bad_alloc &) {
        return GSP_ERR_ALLOC;
    }
    return GSP_OK;
}

const char *gsp_status_string(gsp_status s) {
    switch (s) {
        case GSP_OK: return "GSP_OK";
        case GSP_ERR_INVALID_ARG: return "GSP_ERR_INVALID_ARG";
        case GSP_ERR_TOO_SHORT: return "GSP_ERR_TOO_SHORT";
        case GSP_ERR_ALLOC: return "GSP_ERR_ALLOC";
        case GSP_ERR_CUDA: return "GSP_ERR_CUDA";
        case GSP_ERR_TOO_LARGE: return "GSP_ERR_TOO_LARGE";
    }
    return "GSP_ERR_UNKNOWN";
}

const char *gsp_version(void) { return "libgsp 0.2 (sm_100a)"; }

}  // extern "C"
