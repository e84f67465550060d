/* gsp.h — C ABI of libgsp: B200-native two-stage subband incoherent dedispersion.
 *
 * The operation is the hot path the GSP paper (arXiv 2110.12749) moves to the GPU:
 * PRESTO-style "prepsubband" sub-band dedispersion (§2.3), i.e. the
 * shift-and-sum of Algorithm 1 / Algorithm 2
 * applied twice:
 *
 *   tables (once per plan, host, IEEE binary64, rule R3 = floor(x + 0.5)):
 *     f_c      = f_top + c*chan_bw                      (MHz, c = 0..nchan-1, c=0 highest)
 *     fref_s   = f_{s*cps},  cps = nchan/nsub           (top channel of subband s)
 *     s1[c]    = R3( K*subband_dm*(f_c^-2 - fref_{sub(c)}^-2) / dt )
 *     s2[d][s] = R3( K*dm_list[d]*(fref_s^-2 - f_0^-2) / (dt*downsamp) )
 *     K = 4.148808e3 s MHz^2 pc^-1 cm^3                 (BASELINE.json north_star)
 *   stage 1:   S_s[t]  = sum_{c in subband s} x[t + s1[c]][c],       t in [0, n1)
 *   downsamp:  S'_s[u] = (1/ds) sum_{k<ds} S_s[u*ds + k],            u in [0, n1d)
 *   stage 2:   y_d[u]  = sum_s S'_s[u + s2[d][s]],                   u in [0, nout)
 *   with H1 = max s1, H2 = max s2, n1 = nsamp-H1, n1d = floor(n1/ds), nout = n1d-H2.
 *   (matrices "numpts x numchan" in, "numdm x numpts" out: PAPER.md:102; float32
 *   output: PAPER.md:206; DownSamp: Tables 2-3; readings: DESIGN.md.)
 *
 * Conventions
 *   - No C++ types and no exceptions cross this boundary; every call returns a status.
 *   - "d_" pointers are DEVICE pointers, "h_" pointers are HOST pointers.
 *   - The caller owns d_in/d_out/h_in/h_out and the CUDA stream.  The plan owns its
 *     copies of dm_list, the delay tables (host + device) and the subband workspace;
 *     gsp_plan_destroy frees them.
 *   - gsp_dedisperse only enqueues work on `cuda_stream` (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream) and returns without synchronising.
 *     One plan must not be used from two streams at once (shared workspace), nor from
 *     two host threads at once (launch-time caches on the plan are not locked): a plan is
 *     single-threaded; different plans may be used from different threads freely.
 *   - There is no CPU fallback: without a usable CUDA device plan creation fails
 *     with GSP_ERR_CUDA.
 */
#ifndef GSP_H_
#define GSP_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gsp_plan gsp_plan; /* opaque, heap-owned by the library */

typedef enum { GSP_U8 = 0, GSP_F32 = 1 } gsp_dtype;

typedef enum {
    GSP_OK = 0,
    GSP_ERR_INVALID_ARG = 1, /* null pointer, nchan<1, nsub<1, nchan%nsub!=0, chan_bw>=0,
                                lowest f_c<=0, dt<=0, ndm<1, downsamp<1, negative or
                                non-finite DM, unknown dtype / option                  */
    GSP_ERR_TOO_SHORT = 2,   /* nout <= 0 for this nsamp                                 */
    GSP_ERR_ALLOC = 3,       /* host or device allocation failed                         */
    GSP_ERR_CUDA = 4,        /* CUDA runtime error at create or at launch (launch-time
                                check is cudaPeekAtLastError; asynchronous faults surface
                                at the caller's next synchronisation)                    */
    GSP_ERR_TOO_LARGE = 5    /* gsp_dedisperse_static only: the subband intermediate of this
                                problem does not fit the library's fixed workspace        */
} gsp_status;

/* Kernel implementation selectors for gsp_plan_set_impl (testing / benchmarking). */
typedef enum {
    GSP_IMPL_AUTO = 0,    /* tiled kernels where the plan's shape allows, else generic   */
    GSP_IMPL_GENERIC = 1, /* one thread per output, global loads (Algorithm 2 twice)     */
    GSP_IMPL_TILED = 2,   /* shared-memory staged kernels; INVALID_ARG if unsupported    */
    GSP_IMPL_WINDOWED = 3 /* stage 1 only: the windowed tile kernel for every channel group
                             (TILED streams the groups whose shifts fit its ring and uses
                             the windowed kernel for the rest); INVALID_ARG if unsupported */
} gsp_impl;

/* Build a plan (delay tables per the header comment, device copies, workspace).
 *   nchan      number of frequency channels
 *   f_top      MHz, CENTRE of channel 0 (the highest-frequency channel)
 *   chan_bw    MHz, channel spacing, must be < 0
 *   dt         seconds per input sample
 *   nsamp      input samples (rows of d_in) per gsp_dedisperse call
 *   nsub       number of subbands, must divide nchan
 *   subband_dm pc cm^-3, the DM stage 1 removes inside each subband, >= 0
 *   dm_list    host array of ndm trial DMs (pc cm^-3, >= 0, any order); copied
 *   downsamp   ds >= 1, applied between the stages
 *   in_dtype   element type of d_in
 * On failure *out_plan is set to NULL. */
gsp_status gsp_plan_create(gsp_plan **out_plan, int nchan, double f_top, double chan_bw,
                           double dt, int64_t nsamp, int nsub, double subband_dm,
                           const double *dm_list, int ndm, int downsamp, gsp_dtype in_dtype);

/* Enqueue stage 1 (+downsample) and stage 2 on cuda_stream.
 *   d_in   device, time-major x[t][c], t<nsamp, c<nchan, row pitch = nchan elements of
 *          in_dtype, base address 16-byte aligned
 *   d_out  device, float32 y[d][u], d<ndm (in dm_list order), u<nout, row pitch =
 *          gsp_plan_out_pitch(plan) elements; elements u>=nout of a row are not written;
 *          base address 16-byte aligned; must not alias d_in */
gsp_status gsp_dedisperse(gsp_plan *plan, const void *d_in, float *d_out, void *cuda_stream);

/* gsp_dedisperse for nplans plans over the SAME input, in order: d_outs[i] receives what
 * gsp_dedisperse(plans[i], d_in, d_outs[i], cuda_stream) writes, bit for bit.  This is how the DM ranges of
 * a DDplan run back to back (Tables 2-3 of the paper: one prepsubband pass per range over
 * the same data).  Runs of 2 ... 4 consecutive plans of equal input geometry (nchan, nsamp, nsub) share their
 * stage 1: float32 plans that run the streaming kernel and uint8 plans whose channel groups all run the ring
 * kernel stream the input through ONE shared-memory ring from which every plan gathers with its own shifts
 * (the input is fetched once; the float32 path keeps a per-plan scratch of nchan/16 x nsamp floats: reserve it
 * with gsp_plan_reserve_multi, else the first call that needs it allocates it — a cudaMalloc, which synchronises
 * the device and cannot be captured; when the allocation fails the plans run side by side instead); float32 plans whose shift spreads leave no room for a common ring run side by side in
 * one launch; otherwise the calls are simply made one after the other.  Plans must be distinct.  With stage
 * timing enabled, the times of the shared launches are recorded on plans[0]. */
gsp_status gsp_dedisperse_multi(gsp_plan *const *plans, int nplans, const void *d_in, float *const *d_outs,
                                void *cuda_stream);
/* Allocate now whatever gsp_dedisperse_multi would otherwise allocate on its first call with this plan (float32
 * plans that stream: nchan/16 x nsamp floats rounded up to 32768 columns, about 2 GiB on the 4096-channel, 2^21-
 * sample DDplan workload; nothing for other plans).  The size depends on the plan alone, not on which plans it
 * is later grouped with, so after this call gsp_dedisperse_multi only enqueues.  GSP_ERR_ALLOC when the memory
 * is not there (gsp_dedisperse_multi then still works: it runs the plans side by side). */
gsp_status gsp_plan_reserve_multi(gsp_plan *plan);
/* Kernels one gsp_dedisperse_multi call launches for these plans with their current settings (host, pure). */
int32_t gsp_dedisperse_multi_launches(gsp_plan *const *plans, int nplans);

/* Same result from HOST buffers: h_in[nsamp][nchan] (pinned memory recommended) is copied
 * to the device in time chunks that overlap by the plan's halo, each chunk is dedispersed
 * with the same kernels, and the rows are copied back into h_out[d*h_out_pitch + u].
 * Copies and kernels are pipelined on internal streams; the call returns after the last
 * byte of h_out is written (it synchronises).  cuda_stream orders the start of the work. */
gsp_status gsp_dedisperse_host(gsp_plan *plan, const void *h_in, float *h_out,
                               int64_t h_out_pitch, void *cuda_stream);

/* The same pipeline with the result left on the DEVICE: h_in is a HOST array as above, d_out a DEVICE array
 * y[d][u] of row pitch d_out_pitch >= nout elements, filled exactly as gsp_dedisperse fills it (bit for bit).
 * Only the input crosses PCIe.  This is the call for a pipeline that goes on working on the series on the GPU —
 * dedispersion followed by the single-pulse search: gsp_search_run on d_out, then a copy of
 * the candidate list (bytes, not the gigabytes of time series).  Synchronises like gsp_dedisperse_host. */
gsp_status gsp_dedisperse_host_in(gsp_plan *plan, const void *h_in, float *d_out, int64_t d_out_pitch,
                                  void *cuda_stream);

/* NULL is a no-op returning GSP_OK. */
gsp_status gsp_plan_destroy(gsp_plan *plan);

/* ---- host-side getters (pure, no CUDA work) ---- */
int64_t gsp_plan_nout(const gsp_plan *plan);      /* valid samples per DM row            */
int64_t gsp_plan_out_pitch(const gsp_plan *plan); /* elements between DM rows, >= nout   */
int64_t gsp_plan_halo(const gsp_plan *plan);      /* H1 + ds*H2, raw input samples       */
int64_t gsp_plan_n1(const gsp_plan *plan);        /* nsamp - H1                          */
int64_t gsp_plan_n1d(const gsp_plan *plan);       /* floor(n1/ds)                        */
int32_t gsp_plan_h1(const gsp_plan *plan);        /* max stage-1 shift                   */
int32_t gsp_plan_h2(const gsp_plan *plan);        /* max stage-2 shift                   */
int32_t gsp_plan_ndm(const gsp_plan *plan);
const int32_t *gsp_plan_stage1_shifts(const gsp_plan *plan); /* host, nchan entries      */
const int32_t *gsp_plan_stage2_shifts(const gsp_plan *plan); /* host, ndm*nsub, DM-major,
                                                                in dm_list order         */
int64_t gsp_plan_workspace_bytes(const gsp_plan *plan); /* device bytes owned by the plan */

/* ---- implementation control and instrumentation ---- */
/* stage = 1 or 2.  Returns INVALID_ARG if the requested kernel cannot run this plan. */
gsp_status gsp_plan_set_impl(gsp_plan *plan, int stage, gsp_impl impl);
/* The implementation a stage will actually run (GSP_IMPL_GENERIC, GSP_IMPL_TILED or, for
 * stage 1, GSP_IMPL_WINDOWED). */
int32_t gsp_plan_get_impl(const gsp_plan *plan, int stage);
/* Kernels launched by one gsp_dedisperse call with the current settings. */
int32_t gsp_plan_launches_per_call(const gsp_plan *plan);
/* How the tiled stage 1 splits this plan's channels between its kernels (host, pure):
 * counts[0] 64-channel groups of the channel-major ring kernel, counts[1] / counts[2] subbands of the
 * wide streaming kernel (two / one CTA per SM), counts[3] 64-channel groups of the windowed kernel,
 * counts[4] 1 when float32 input streams through the time-major ring kernel (0: tile kernel),
 * counts[5] / counts[6] subbands of the ring kernel's long-ring instantiation (one CTA per subband; rings
 * that leave room for two CTAs per SM / larger rings). */
gsp_status gsp_plan_stage1_split(const gsp_plan *plan, int32_t counts[7]);
/* The same counts, sized by the caller: writes the first min(ncounts, GSP_STAGE1_SPLIT_COUNTS) entries and
 * nothing past counts[ncounts-1]; *navailable (optional) receives how many the library has.  Use this one:
 * the fixed-size call above wrote 5 entries in libgsp 0.1 and writes 7 since 0.2, so a caller compiled
 * against the older header is overrun.  Diagnostic arrays added later will grow this list, never the
 * fixed-size call (gsp_version tells the builds apart). */
#define GSP_STAGE1_SPLIT_COUNTS 7
gsp_status gsp_plan_stage1_split_n(const gsp_plan *plan, int32_t *counts, int32_t ncounts, int32_t *navailable);
/* When enabled, every gsp_dedisperse call records CUDA events on its stream around each
 * stage (no synchronisation).  Enabling (again) clears the recorded calls. */
gsp_status gsp_plan_enable_stage_timing(gsp_plan *plan, int enable);
/* Device time of the LAST timed call's stages in milliseconds; synchronises on its events.
 * INVALID_ARG if timing is disabled or no call was made. */
gsp_status gsp_plan_last_stage_ms(gsp_plan *plan, float *ms_stage1, float *ms_stage2);
/* Sum over all calls recorded since timing was enabled: total stage-1 ms, total stage-2 ms
 * and the number of calls; synchronises on the last call's events. */
gsp_status gsp_plan_stage_ms_total(gsp_plan *plan, double *ms_stage1, double *ms_stage2,
                                   int32_t *ncalls);

/* ---- pure host helpers (no CUDA device needed) ---- */
/* The plan's delay-table builder on its own: s1[nchan], s2[ndm*nsub] (DM-major, dm_list
 * order), rule R3 of the header comment.  Same argument checks as gsp_plan_create. */
gsp_status gsp_delay_tables(int nchan, double f_top, double chan_bw, double dt, int nsub,
                            double subband_dm, const double *dm_list, int ndm, int downsamp,
                            int32_t *s1, int32_t *s2);

/* ---- RFI prologue (the pipeline step before dedispersion), uint8 plans ----
 * "pulsar search (RFI mitigation, de-dispersion and single-pulse search)"; the 'mask' and 'clip'
 * options of prepsubband.  The paper prints no mechanics; the operation is readings F1-F4 of
 * DESIGN.md 3a, in exact integers and one binary64 comparison so that it has exactly one result:
 *   F1 x1[t][c] = chan_mask[c] ? chan_pad[c] : x[t][c]
 *   F2 z[t] = sum_c x1[t][c]                                   (the zero-DM series)
 *   F3 per block of clip_block rows (n rows in the ragged last block): S1 = sum z, S2 = sum z^2; row t is
 *      clipped iff (double)(n*z[t] - S1) > clip_sigma * sqrt((double)(n*S2 - S1*S1))
 *   F4 x2[t][c] = clipped[t] ? chan_pad[c] : x1[t][c]; gsp_dedisperse then computes its result from x2.
 * h_chan_mask: nchan bytes, non-zero = masked, or NULL (no mask); h_chan_pad: nchan bytes (both HOST, copied).
 * clip_sigma = 0 disables the clip; otherwise clip_block must be a multiple of 32 in [32, 8192] with
 * clip_block * nchan * 255 < 2^31.  The replacement is applied inside the stage-1 kernels (no pass over the
 * input is added); the clip adds one read of the input for the zero-DM statistics.  h_chan_pad = NULL removes
 * the prologue.  Which stage-1 kernels carry it: the ring kernel and its long-ring instantiations, and the generic
 * one-thread-per-output kernel.  A plan keeps its channel groups on the ring kernels and runs only the subbands
 * that would need the wide or the windowed kernel (very wide shift spreads) through the generic kernel, in one
 * extra launch; a plan the ring kernels cannot take at all (fewer than 16 channels per subband, nchan not a
 * multiple of 64, one-stage plans) runs its whole stage 1 on the generic kernel — correct, but many times
 * slower; gsp_plan_get_impl(plan, 1) and gsp_plan_stage1_split_n tell which case a plan is in.
 * INVALID_ARG for float32 plans, for gsp_dedisperse_host on a plan with a prologue (clip blocks
 * are defined on the whole input) and when a forced stage-1 kernel has no prologue. */
gsp_status gsp_plan_set_rfi(gsp_plan *plan, const uint8_t *h_chan_mask, const uint8_t *h_chan_pad,
                            double clip_sigma, int32_t clip_block);
/* Diagnostics of the LAST gsp_dedisperse call of a clipping plan (synchronises the device): the zero-DM
 * series z[nsamp] and the per-row clip flags [nsamp] (either pointer may be NULL), HOST arrays. */
gsp_status gsp_plan_rfi_last(const gsp_plan *plan, int64_t *h_zero_dm, uint8_t *h_clipped);

/* ---- single-pulse search on the dedispersed series (the pipeline step after dedispersion) ----
 * "pulsar search (RFI mitigation, de-dispersion and single-pulse search)"; the paper runs this
 * step on the CPU and prints no mechanics, so the operation is the set of readings S1-S6 of
 * DESIGN.md 3a, taken in stated precisions so that it has exactly one result:
 *   S1 blocks of `block` samples per DM row (last block ragged, n samples); S1 = sum y, S2 = sum y^2 in
 *      binary64, added in a perfect binary tree over the block's slots in natural order (absent slots = 0)
 *   S2 mu = S1/n, var = S2/n - mu*mu (no FMA), r = var > 0 ? 1/sqrt(var) : 0; mu_f, r_f = float32 roundings
 *   S3 z[u] = (y[u] - mu_f) * r_f in float32, each sample with its own block's statistics
 *   S4 boxcars of widths 2^j, j < nwidths: B_0 = z, B_{j+1}[u] = B_j[u] + B_j[u + 2^j] (float32), valid while
 *      u + 2^j <= nout; snr_j[u] = B_j[u] * c_j, c_j = 2^(-j/2) as float32 (1, 0.70710678f, 0.5, 0.35355339f, ...)
 *   S5 per (DM, block): the best (snr, j, u) — larger snr, then smaller j, then smaller u
 *   S6 it is a candidate iff snr >= threshold; candidates are listed in (DM, block) order.
 * A constant block (var = 0) has r_f = 0, hence z = 0 on all of it: its width-1 snr is exactly 0, and a boxcar
 * that starts in it and reaches into block b+1 takes that block's normalised values.  Its winner is therefore
 * (snr 0, width 1, first sample of the block) unless such a reaching boxcar is positive; it is listed like any
 * other winner iff snr >= threshold (so: never for a positive threshold unless a pulse sits right behind the
 * block's end, always for threshold <= 0).
 * The input must be finite.  NaN / Inf samples are outside the definition: the library's and the oracle's
 * comparisons treat NaN differently and (float)r can overflow, so neither result is specified. */
typedef struct gsp_search gsp_search; /* opaque, heap-owned by the library */

/* ndm rows of nout valid samples at row pitch `pitch` elements (>= nout, a multiple of 4: what
 * gsp_plan_out_pitch returns); block in {256, 512, 1024, 2048}; 1 <= nwidths <= 6 (widths 1 ... 32);
 * max_cand = capacity of the caller's candidate arrays (0: count only).  On failure *out is NULL. */
gsp_status gsp_search_create(gsp_search **out, int ndm, int64_t nout, int64_t pitch, int block, int nwidths,
                             float threshold, int64_t max_cand);
/* Enqueue the search of d_y[ndm][pitch] (device, float32, 16-byte aligned: the d_out of gsp_dedisperse) on
 * cuda_stream; no synchronisation.  Device outputs: *d_count = number of candidates found (it may exceed
 * max_cand; only the first max_cand, in (DM, block) order, are stored), d_cand_dm / d_cand_sample /
 * d_cand_width (int32) and d_cand_snr (float32), max_cand entries each.  d_stats is optional (NULL): when
 * given it receives (mu_f, r_f) of every block, [ndm][nblocks][2] float32. */
gsp_status gsp_search_run(gsp_search *search, const float *d_y, int32_t *d_cand_dm, int32_t *d_cand_sample,
                          int32_t *d_cand_width, float *d_cand_snr, int64_t *d_count, float *d_stats,
                          void *cuda_stream);
int64_t gsp_search_nblocks(const gsp_search *search); /* blocks per DM row */
gsp_status gsp_search_destroy(gsp_search *search);    /* NULL is a no-op returning GSP_OK */

/* ---- dedispersion that allocates nothing (for callers that cannot call cudaMalloc) ----
 * Who needs it: a real-time recording backend whose other streams must not be stalled by the device-wide
 * synchronisation that cudaMalloc / cudaFree imply; a process whose device memory was handed out in full at
 * start-up (a framework's pool, a fixed arena), where an allocation made behind the owner's back fails or
 * eats memory the owner counted on; any code past a "no allocation after initialisation" line.  A gsp_plan
 * allocates when it is created, so such callers cannot hold one.  This call needs no plan and makes no
 * cudaMalloc, cudaFree or allocating library call, on the first call or any later one.
 *
 * It computes exactly what gsp_dedisperse computes (stage 1, downsample, stage 2 of the header comment;
 * Algorithm 2 of the paper applied twice) with one thread per output.  The caller passes
 * every input and the output; the subband intermediate S'[nsub][n1d] lives in a fixed array inside the
 * library image.  LIMIT: nsub * n1d * 4 bytes <= GSP_STATIC_WS_BYTES (16 MiB, i.e. 4 Mi subband samples,
 * e.g. 64 subbands x 65536 samples); a larger problem returns GSP_ERR_TOO_LARGE before any GPU work — split
 * it into time blocks that overlap by the halo h1 + downsamp*h2.  COST: every GPU on which the library's
 * code is loaded holds those 16 MiB until the process exits, whether or not this call is ever made.
 *
 *   d_in       device, x[nsamp][nchan] of in_dtype, time-major, as for gsp_dedisperse
 *   d_s1       device, int32 [nchan]       stage-1 shifts   } build both on the host with gsp_delay_tables
 *   d_s2       device, int32 [ndm][nsub]   stage-2 shifts   } (no CUDA call) and copy them into your memory
 *   h1, h2     HOST values: the largest entry of s1 and of s2.  They fix n1 = nsamp - h1,
 *              n1d = floor(n1/downsamp), nout = n1d - h2.  Values smaller than the true maxima make the
 *              kernels read past the end of d_in; the tables live on the device, so this is not checked.
 *   d_out      device, float32 y[d][u], u < nout, row pitch out_pitch >= nout elements; u >= nout untouched
 *   cuda_stream  the work is enqueued here without synchronising; the stream's device must be current
 * Errors: INVALID_ARG (null pointer, bad sizes, nsub or ndm > 65535, nchan/nsub or nsub > 12288,
 * out_pitch < nout), TOO_SHORT (nout <= 0), TOO_LARGE (above), CUDA (runtime error).
 *
 * Set-up: the first call on each device asks the CUDA runtime once for the array's device address
 * (cudaGetSymbolAddress; this loads the module on that device, it does not allocate).  Make that first call
 * during your own set-up, before you start capturing any stream.
 * Sharing: all calls on one device use the same array, and it keeps whatever the last call left in it.
 * Nothing in it needs to start at zero — stage 1 overwrites every element that stage 2 reads — so a call is
 * not affected by the one before it.  But two calls that can overlap on the GPU (different streams without an
 * ordering between them, or two threads) overwrite each other's intermediate and both produce garbage: order
 * every call on a device after the previous one.  Calls on different devices are independent. */
#define GSP_STATIC_WS_BYTES (16u << 20)
gsp_status gsp_dedisperse_static(const void *d_in, gsp_dtype in_dtype, int64_t nsamp, int nchan, int nsub,
                                 int ndm, int downsamp, const int32_t *d_s1, const int32_t *d_s2,
                                 int32_t h1, int32_t h2, float *d_out, int64_t out_pitch, void *cuda_stream);
int64_t gsp_static_workspace_bytes(void); /* GSP_STATIC_WS_BYTES, for callers without the header */

const char *gsp_status_string(gsp_status status);
const char *gsp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GSP_H_ */
