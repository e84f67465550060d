// gsp_internal.h — private declarations shared by the libgsp translation units.
// (Nothing here is visible through include/gsp.h; the oracle never includes it.)
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "gsp.h"

namespace gsp {

// ----------------------------------------------------------------------------------
// Workspace formats of the subband intermediate S' (written by stage 1, read by stage 2)
// ----------------------------------------------------------------------------------
enum WsFormat : int {
    WS_I32 = 0,   // int32  S'[s][ws_pitch]   un-divided ds-sum (uint8 input: generic stage 2, and the tiled
                  //                          stage 2 when the sums exceed 16 bits)
    WS_F32 = 1,   // float  S'[s][ws_pitch]   un-divided ds-sum (float32 input)
    WS_PK16 = 2,  // uint32 W[s][ws_pitch]    W[i] = S'[i] | S'[i+M] << 16  (uint8 input, tiled
                  //                          stage 2; M = plane length)
};

// Operand format / fold schedule of the tiled stage-2 kernel.
enum Stage2Mode : int {
    S2_PK4 = 0,   // packed u16 pairs, four subbands summed in 16-bit lanes between folds (4*cps*255*ds <= 65535)
    S2_PK2 = 1,   // packed u16 pairs, two subbands between folds
    S2_PK1 = 2,   // packed u16 pairs, folded after every subband (cps*255*ds <= 65535)
    S2_I32 = 3,   // int32 operands, one per word (larger un-divided sums: high DownSamp)
    S2_F32 = 4,   // float32 operands
};

// Geometry of the tiled stage-2 kernel, fixed at plan creation.
struct Stage2Tiling {
    bool supported = false;
    int mode = S2_PK4;
    int Q = 0;            // DM trials per CTA tile
    int M = 0;            // words per tile row; a tile covers T = tpw*M output samples
    int tpw = 2;          // output samples per 32-bit word: 2 (packed u16 pairs) or 1 (float32)
    int chunk = 4;        // subbands per pipeline stage (= flush interval of the u16x2 sums)
    int nchunk = 0;       // nsub / chunk
    int nstage = 0;       // pipeline depth
    int stage_words = 0;  // 32-bit words per stage buffer
    int ndmblk = 0;       // ceil(ndm / Q)
    int64_t ntile_t = 0;  // ceil(nout / (2*M))
    size_t smem_bytes = 0;
};

// A tensor map of the caller's input, cached per kernel family and re-encoded only when d_in or the box
// geometry changes.  The cache is launch-time state of the plan: a plan is used by one thread at a time (gsp.h).
struct TmapCache {
    const void *d_in = nullptr;
    int box_chan = 0, box_rows = 0, swizzle_bytes = 0;   // the whole key: a slot reused with another box re-encodes
    bool valid = false;
    alignas(64) CUtensorMap tm;
};
enum TmapSlot : int { TMAP_RING = 0, TMAP_WIDE = 1, TMAP_F32 = 2, TMAP_LONG = 3, TMAP_SPLIT = 4, TMAP_COUNT = 5 };

constexpr int kRingMaxPlans = 4;   // plans that can share the uint8 ring of one stage-1 launch
constexpr int kLongLists = 3;      // launches of the long-ring instantiations of the uint8 ring kernel

// RFI prologue of a plan (gsp_plan_set_rfi): channel mask + pad values, block-wise zero-DM clip.
struct RfiState {
    bool enabled = false;
    bool has_mask = false;
    double clip_sigma = 0.0;        // 0: no clipping
    int clip_block = 0;             // rows per statistics block
    uint8_t *d_mask = nullptr;      // [nchan] 1 = masked (nullptr: none)
    uint8_t *d_pad = nullptr;       // [nchan]
    uint8_t *d_keep = nullptr;      // [nchan] 1 - mask (dp4a weights of the zero-DM sum)
    int32_t *d_z = nullptr;         // [nsamp] zero-DM series of the last call
    uint32_t *d_clip_bits = nullptr;   // bit t: row t clipped (padded past nsamp with zeros)
    int64_t pad_sum = 0;            // sum of the pad values of the masked channels
    // subbands none of the ring kernels takes (wide / windowed groups): with a prologue they run the generic
    // kernel, the rest of the plan stays on the ring kernels
    int32_t *d_rest = nullptr;
    int nrest = 0;
};

struct HostStream;  // gsp_stage1_wide.cu — streaming stage 1 for uint8 subbands with large shift spreads
bool stage1_wide_supported(const gsp_plan &p);
int stage1_wide_slots(const gsp_plan &p, int s);
int stage1_wide_mid_slots();
cudaError_t configure_stage1_wide(const gsp_plan &p);
cudaError_t launch_stage1_wide(const gsp_plan &p, const void *d_in, cudaStream_t st);

// gsp_stage1_f32.cu — tiled stage 1 for float32 input
bool stage1_f32_supported(const gsp_plan &p);
void plan_stage1_f32(gsp_plan &p);            // decide (once) whether the streaming kernel runs this plan
bool stage1_f32_streams(const gsp_plan &p);   // the streaming kernel (not the tile kernel) runs this plan
cudaError_t configure_stage1_f32(const gsp_plan &p);
cudaError_t launch_stage1_f32(const gsp_plan &p, const void *d_in, cudaStream_t st);
// several plans over the same float32 input in one launch of the streaming kernel (gsp_dedisperse_multi)
bool stage1_f32_multi_ok(gsp_plan *const *plans, int np);
cudaError_t launch_stage1_f32_multi(gsp_plan *const *plans, int np, const void *d_in, cudaStream_t st);
int stage1_f32_multi_launches(gsp_plan *const *plans, int np);
cudaError_t reserve_stage1_f32_shared(gsp_plan &p);   // gsp_plan_reserve_multi: the shared-ring scratch, up front

// gsp_host.cu

}  // namespace gsp

struct gsp_plan {
    // ---- arguments ----
    int nchan = 0, nsub = 0, cps = 0, ndm = 0, ds = 1;
    double f_top = 0, chan_bw = 0, dt = 0, subband_dm = 0;
    int64_t nsamp = 0;
    gsp_dtype dtype = GSP_U8;
    std::vector<double> dm_list;

    // ---- tables and extents (host) ----
    std::vector<int32_t> s1;        // [nchan]
    std::vector<int32_t> s2;        // [ndm][nsub], dm_list order
    std::vector<int32_t> order;     // sorted position -> dm_list row
    int32_t H1 = 0, H2 = 0;
    int64_t n1 = 0, n1d = 0, nout = 0, out_pitch = 0, halo = 0;

    // ---- device state ----
    int device = 0;
    int sm_count = 0;
    size_t smem_optin = 0;          // cudaDevAttrMaxSharedMemoryPerBlockOptin of the device
    int32_t *d_s1 = nullptr;        // [nchan]
    int32_t *d_s2 = nullptr;        // [ndm][nsub] dm_list order (generic stage 2)
    void *d_ws = nullptr;           // subband workspace
    size_t ws_bytes = 0;
    int64_t ws_pitch = 0;           // elements per subband row of the workspace
    gsp::WsFormat ws_format = gsp::WS_I32;

    // tiled stage 1: 64-channel groups run the streaming ring kernel (gsp_stage1_ring.cu) when their
    // largest shift fits its ring, else the windowed tile kernel (gsp_stage1.cu)
    std::vector<int32_t> g_ring;    // groups of the streaming ring kernel
    std::vector<int32_t> g_win;     // groups of the windowed kernel
    std::vector<int32_t> g_all;     // every group (windowed kernel forced for all)
    int32_t *d_g_ring = nullptr;
    int32_t *d_g_win = nullptr;
    int32_t *d_g_all = nullptr;
    // subbands of the wide streaming kernel (gsp_stage1_wide.cu): [0] two CTAs per SM, [1] one CTA per SM
    std::vector<int32_t> s_wide[2];
    int32_t *d_s_wide[2] = {nullptr, nullptr};
    int ns_wide[2] = {0, 0};        // ring slots of each list
    // subbands of the LONG instantiations of the ring kernel (one CTA per subband, ring length per launch):
    // [0] common stream, two CTAs per SM; [1] per-slice streams, two CTAs per SM; [2] per-slice streams, one
    std::vector<int32_t> u_long[gsp::kLongLists];
    int32_t *d_u_long[gsp::kLongLists] = {nullptr, nullptr, nullptr};
    int rl_long[gsp::kLongLists] = {0, 0, 0};        // ring rows of each launch
    int nst_long[gsp::kLongLists] = {0, 0, 0};       // TMA stages of each launch
    int64_t seg_long[gsp::kLongLists] = {0, 0, 0}, nseg_long[gsp::kLongLists] = {0, 0, 0};   // S-samples per CTA time segment, segments
    int f32_slots = 0;              // ring slots of the float32 streaming kernel (0: the tile kernel runs)
    float *d_f32_part = nullptr;    // shared-ring path of gsp_dedisperse_multi: partial sums of the 16-channel
    size_t f32_part_bytes = 0;      // groups, [nchan / 16][pitch] float32 (allocated on first use)
    int64_t ring_seg_rows = 0;      // S-samples per CTA time segment of the ring kernel
    int64_t ring_nseg = 0;

    // tiled stage 2
    gsp::Stage2Tiling t2;
    int4 *d_t2_prod = nullptr;      // [ndmblk][nsub] {window start, window words, buffer offset, 0}
    int32_t *d_t2_offs = nullptr;   // [ndmblk*Q][nsub] word offset of W_s[u0 + s2[d][s]] in its stage
    int32_t *d_t2_rows = nullptr;   // [ndmblk*Q] output row of sorted DM d, or -1 (padding)

    // ---- implementation selection ----
    int req_impl[3] = {0, GSP_IMPL_AUTO, GSP_IMPL_AUTO};
    int impl[3] = {0, GSP_IMPL_GENERIC, GSP_IMPL_GENERIC};

    // ---- instrumentation ----
    bool timing = false;
    std::vector<cudaEvent_t> ev;    // 3 events per recorded call: start, after stage 1, end
    size_t ev_used = 0;             // events in use (multiple of 3)

    // ---- cached tensor maps of the caller's input (launch-time state, hence mutable) ----
    mutable gsp::TmapCache tmaps[gsp::TMAP_COUNT];

    // ---- RFI prologue ----
    gsp::RfiState rfi;

    // ---- host-buffer streaming (lazy) ----
    gsp::HostStream *hs = nullptr;
};

namespace gsp {

// gsp_tables.cpp — host-only arithmetic (no CUDA calls)
gsp_status validate_args(int nchan, double f_top, double chan_bw, double dt, int64_t nsamp,
                         int nsub, double subband_dm, const double *dm_list, int ndm,
                         int downsamp, int in_dtype);
void build_delay_tables(gsp_plan &p);
gsp_status compute_extents(gsp_plan &p);
void plan_stage2_tiling(gsp_plan &p, size_t smem_budget_bytes);
// host images of the tiled stage-2 tables
void build_stage2_tables(const gsp_plan &p, std::vector<int4> &prod, std::vector<int32_t> &offs,
                         std::vector<int32_t> &rows);

// gsp_kernels.cu — launchers (enqueue only)
cudaError_t launch_stage1_generic(const gsp_plan &p, const void *d_in, cudaStream_t st);
// the same kernel for the nlist subbands of a device list only (RFI plans: the subbands outside the ring kernels)
cudaError_t launch_stage1_generic_list(const gsp_plan &p, const void *d_in, const int32_t *d_list, int nlist,
                                       cudaStream_t st);
cudaError_t launch_stage2_generic(const gsp_plan &p, float *d_out, cudaStream_t st);
cudaError_t launch_stage2_tiled(const gsp_plan &p, float *d_out, cudaStream_t st);
cudaError_t configure_kernels(const gsp_plan &p);

// gsp_stage1.cu — tiled stage 1
bool stage1_tiled_supported(const gsp_plan &p);
cudaError_t configure_stage1(const gsp_plan &p);
// groups: device list of 64-channel group indices to process (ngroups entries)
cudaError_t launch_stage1_tiled(const gsp_plan &p, const void *d_in, const int32_t *d_groups, int ngroups,
                                cudaStream_t st);

// one-stage plans (nsub == nchan): stage 1 is a transposition into the stage-2 operand format
bool stage1_transpose_supported(const gsp_plan &p);
cudaError_t launch_stage1_transpose(const gsp_plan &p, const void *d_in, cudaStream_t st);

// gsp_stage1_ring.cu — streaming stage 1
bool stage1_ring_supported(const gsp_plan &p);
void plan_stage1_groups(gsp_plan &p);
cudaError_t configure_stage1_ring(const gsp_plan &p);
cudaError_t launch_stage1_ring(const gsp_plan &p, const void *d_in, cudaStream_t st);
cudaError_t launch_stage1_ring_long(const gsp_plan &p, const void *d_in, cudaStream_t st);
// several uint8 plans over the same input sharing ONE ring (gsp_dedisperse_multi)
bool stage1_ring_multi_ok(gsp_plan *const *plans, int np);
cudaError_t launch_stage1_ring_multi(gsp_plan *const *plans, int np, const void *d_in, cudaStream_t st);
// tensor map of the caller's input {nchan, nsamp} with boxes of box_chan x box_rows elements (cached on the plan)
cudaError_t input_map(const gsp_plan &p, int slot, const void *d_in, int box_chan, int box_rows, int swizzle_bytes,
                      const CUtensorMap **tm);
bool tma_available();

// gsp_rfi.cu — RFI prologue (channel mask, zero-DM clip)
gsp_status rfi_configure(gsp_plan &p, const uint8_t *h_mask, const uint8_t *h_pad, double clip_sigma, int clip_block);
void rfi_free(RfiState &r);
cudaError_t launch_rfi_prepass(const gsp_plan &p, const void *d_in, cudaStream_t st);
gsp_status rfi_read_back(const gsp_plan &p, int64_t *h_z, uint8_t *h_clipped);

// gsp_host.cu
gsp_status host_dedisperse(gsp_plan *plan, const void *h_in, float *h_out, int64_t h_out_pitch,
                           cudaStream_t st, bool out_on_device = false);
void host_stream_destroy(HostStream *hs);

}  // namespace gsp
