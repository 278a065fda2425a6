// Internal declarations shared by nsfrb_api.cu (plan, C ABI) and nsfrb_kernels.cu (sm_100a
// kernels).  Nothing here is part of the public ABI (include/nsfrb.h) and nothing here is
// shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/nsfrb.h"

namespace nsfrb {

// Per-(pixel, DM group, width batch) result of the search kernel, reduced per pixel by
// k_finalize.  k/j are ORIGINAL indices into dm_list/width_list; snr = -inf, k = -1 when the
// slice defined no cell.  mu/sigma describe the winning series in workspace units (the
// per-channel baseline is already removed), blk is the time block that produced the maximum
// (-1: unknown, rescan everything).
struct Partial {
    float snr;
    int32_t k;
    int32_t j;
    int32_t blk;
    float mu;
    float sigma;
    int32_t u; // index into the unique-trial tables
    int32_t pad;
};

constexpr int kBlockLen = 256;   // dedispersed samples per time block (8 per lane)
constexpr int kWidthBatch = 32;  // widths one search CTA tracks in registers
constexpr int kSearchWarps = 16; // warps per search CTA = DM trials held on chip per CTA
constexpr int kStageStride = 288; // floats per trial in the dedispersion staging tile: t + 4*(t>>5), t < 256

struct SearchParams {
    const float *W;          // [npix][nchan][pitch]  time-contiguous, baseline removed
    const int32_t *delays_u; // [nuniq][nchan]        unique trials, sorted by dmax
    const int32_t *dmax_u;   // [nuniq]
    const int32_t *k_of_u;   // [nuniq]               lowest original dm index of the trial
    const int32_t *widths;   // [nw]
    const int32_t *dd_tab;   // dedispersion change lists, one record stream per group (see build_dd_tables)
    const int32_t *dd_off;   // [n_groups+1] offsets into dd_tab
    Partial *partials;       // [npix][n_groups*n_wb]
    int32_t npix, nchan, pitch;
    int32_t ring_L;      // slots per (pixel, channel) row = plan nt
    int32_t origin;      // slot of relative raw sample 0
    int32_t len;         // valid raw samples (nt offline; min(n, L) streaming)
    int32_t raw_end_min; // S5: windows must end (raw frame) at or after this relative index
    int32_t nuniq, nw, n_groups, n_wb;
    int32_t H;           // prefix history per series (multiple of 32, >= wmax + kBlockLen + 32)
    int32_t tab_cap;     // ints reserved in shared memory for one group's change lists (multiple of 4)
    int32_t RS;          // raw block row stride in floats
    int32_t wmax;
};

struct StreamState;
struct Search4State;

struct FinalParams {
    const float *W;
    const int32_t *delays_u;
    const int32_t *dmax_u;
    const int32_t *widths;    // [nw_used]
    const int32_t *j_of_used; // [nw_used] original width index
    const Partial *partials;
    float *snr_map;   // [npix]
    int32_t *argmax;  // [3][npix]
    int32_t npix, nchan, pitch, ring_L, origin, len, raw_end_min, slices;
    int32_t t_offset; // added to the reported t (streaming: lo mod 2^31)
};

} // namespace nsfrb

// The plan: host tables + device workspace.  Opaque to callers (include/nsfrb.h).
struct nsfrb_plan {
    int nx = 0, ny = 0, npix = 0, nchan = 0, nt = 0, ndm = 0, nw = 0;
    double tsamp = 0;
    float threshold = 0;
    std::vector<double> freqs, dms;
    std::vector<int32_t> widths;
    std::vector<int32_t> delays; // [ndm][nchan]
    std::vector<int32_t> dmax;   // [ndm]
    // unique trials, sorted by (dmax, first original index)
    int nuniq = 0;
    std::vector<int32_t> k_of_u, dmax_u, delays_u;
    // widths that can hold at least one cell for some trial, original order
    int nw_used = 0;
    std::vector<int32_t> widths_used, j_of_used;
    std::vector<int32_t> stream_worder; // indices into widths_used, ascending width (k_stream's W_TAB order)
    int wmax_used = 0, dmax_all = 0, dmin_all = 0;
    int n_groups = 0, n_wb = 0, H = 0, RS = 0, pitch = 0, tab_cap = 0;
    std::vector<int32_t> dd_tab, dd_off; // per-group dedispersion change lists
    size_t smem_search = 0, smem_final = 0;
    int64_t cells_per_pixel = 0, shift_adds_per_pixel = 0;
    // device
    float *d_W = nullptr;
    int32_t *d_dd_tab = nullptr, *d_dd_off = nullptr;
    int32_t *d_delays_u = nullptr, *d_dmax_u = nullptr, *d_k_of_u = nullptr, *d_widths = nullptr, *d_j_of_used = nullptr;
    nsfrb::Partial *d_partials = nullptr;
    size_t workspace_bytes = 0;
    // streaming state
    int64_t n_received = 0;
    // host-variant staging
    float *d_in = nullptr;
    size_t d_in_bytes = 0;
    float *d_snr = nullptr;
    int32_t *d_arg = nullptr;
    nsfrb_cand *d_cands = nullptr;
    uint32_t d_cands_cap = 0;
    uint32_t *d_ncands = nullptr;
    int last_launches = 0;
    int device = 0;
    // optional per-kernel timing
    bool profiling = false;
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    bool ev_valid = false;
    // real-time path (nsfrb_stream.cu): ring, provisional means, plan-specialised kernel
    nsfrb::StreamState *stream = nullptr;
    float *cube_snr = nullptr;   // caller's optional cube outputs of the real-time path (nsfrb_stream_set_cubes)
    int32_t *cube_toa = nullptr;
    float run_alpha = 0.f;       // running-sigma mode (nsfrb_stream_set_running_sigma): caller's outputs, or null = off
    float *run_snr = nullptr;
    int32_t *run_arg = nullptr;
    // offline path: plan-specialised k_search4 (nsfrb_search_kernel.cuh) + its pixel-batch workspaces (nsfrb_offline.cu)
    nsfrb::Search4State *search4 = nullptr;
    // pipelined host-buffer pushes (nsfrb_stream_push_host_async): two staging slots, a copy and a compute stream
    struct HostPipe {
        cudaStream_t s_copy = nullptr, s_comp = nullptr;
        cudaEvent_t copied[2] = {nullptr, nullptr}, done[2] = {nullptr, nullptr};
        bool busy[2] = {false, false};
        float *d_in[2] = {nullptr, nullptr};
        size_t in_bytes[2] = {0, 0};
        float *d_snr[2] = {nullptr, nullptr};
        int32_t *d_arg[2] = {nullptr, nullptr};
        nsfrb_cand *d_cands[2] = {nullptr, nullptr};
        uint32_t cands_cap[2] = {0, 0};
        uint32_t *d_ncands[2] = {nullptr, nullptr};
        uint64_t count = 0;
    } *pipe = nullptr;
    // candidate selection (nsfrb_cluster.cu): per-CTA key lists + ticket, allocated at the first nsfrb_cluster
    void *d_cluster_ws = nullptr;
};

namespace nsfrb {

// sets the thread-local error text of nsfrb_last_error and returns `code` (for entry points outside nsfrb_api.cu)
int api_fail(int code, const std::string &msg);
int plan_host_init(nsfrb_plan **out, int nx, int ny, int nchan, int nt, const double *freqs_GHz, double tsamp_s,
                   const double *dm_list, int ndm, const int32_t *width_list, int nwidth, float threshold);
void free_plan(nsfrb_plan *p);

// ---- plan-specialised offline kernel and its batch pipeline (nsfrb_offline.cu)
// True if the plan can use k_search4 (at most 32 usable widths, tiles fit shared memory; NSFRB_SEARCH_JIT=0 forces the
// generic k_search).
bool search4_usable(const nsfrb_plan *pl);
int search4_source(const nsfrb_plan *pl, std::string &src, std::string &err);
int search4_prepare(nsfrb_plan *pl, std::string &err); // compile + workspaces; idempotent
// layout change + one launch per pixel batch; the kernels write snr_map/argmax (fused a6).  ev_layout (may be null) is
// recorded after the first batch's layout kernel.
int search4_launch(nsfrb_plan *pl, const float *cube, cudaStream_t st, float *snr_map, int32_t *argmax, int *launches,
                   cudaEvent_t ev_layout, std::string &err);
// the same from a host cube: strided H2D copies of one batch at a time on a copy stream, overlapped with the search
int search4_launch_host(nsfrb_plan *pl, const float *cube_host, cudaStream_t st, float *snr_map, int32_t *argmax, int *launches,
                        std::string &err);
void search4_free(nsfrb_plan *p);
size_t search4_bytes(const nsfrb_plan *p);
int search4_ring_len(const nsfrb_plan *pl);

// ---- real-time path (nsfrb_stream.cu)
void stream_free(nsfrb_plan *p);
void stream_reset(nsfrb_plan *p);
int stream_prepare(nsfrb_plan *pl, int chunk_nt, std::string &err); // allocate + compile ahead of the first push
int stream_set_cubes(nsfrb_plan *pl, float *snr_cube, int32_t *toa_cube, std::string &err);
int stream_set_running(nsfrb_plan *pl, double alpha, float *snr_run, int32_t *arg_run, std::string &err);
size_t stream_bytes(const nsfrb_plan *p); // device bytes the real-time path holds (0 before the first push)
int stream_mode(const nsfrb_plan *p);     // 0 none yet, 1 raw ring, 2 + dedispersed history, 3 + its 8-sample block sums
// a8 + k_stream passes + reduction over slices; outputs as nsfrb_stream_push.  Returns an NSFRB_* code and
// leaves the message in `err`.
int stream_push(nsfrb_plan *pl, const float *chunk, int chunk_nt, cudaStream_t st, float *snr_map, int32_t *argmax,
                int *launches, std::string &err);
// Source text (prologue + kernel) and cubin of the plan's k_stream for a first chunk of chunk_nt samples;
// no CUDA device needed.  `variant` = "" for the default tile shape or "KK,GPC,SEG,TT,MINB".
int stream_source(const nsfrb_plan *pl, int chunk_nt, const char *variant, std::string &src, std::string &err);
int stream_compile(const std::string &src, std::vector<char> &cubin, std::string &log);


// W[p - p_begin][c][t] = cube[c][t][p] - cube[c][0][p] for p in [p_begin, p_begin + p_count)
cudaError_t launch_transpose(const float *cube, float *W, int npix, int nchan, int nt, int pitch, int p_begin, int p_count,
                             cudaStream_t st);
cudaError_t launch_search(const SearchParams &p, size_t smem_bytes, cudaStream_t st);
cudaError_t launch_finalize(const FinalParams &p, size_t smem_bytes, cudaStream_t st);
cudaError_t launch_compact(const float *snr_map, const int32_t *argmax, int npix, float threshold,
                           nsfrb_cand *cands, uint32_t cap, uint32_t *ncands, cudaStream_t st);
cudaError_t launch_bin(const float *in, float *out, int nchan, int nt, long long npix, int factor, cudaStream_t st);
// out may alias in; med ([nchan][npix]) may be null; nt <= median_max_nt()
cudaError_t launch_median(const float *in, float *out, float *med, int nchan, int nt, long long npix, cudaStream_t st);
int median_max_nt();
cudaError_t launch_psf_mask(const float *psf, long long n, long long lo, double frac, uint8_t *mask, double *value,
                            cudaStream_t st);
int cluster_max_top();
int cluster_grid(int npix);
// ws: cluster_grid(npix) * topn 64-bit keys; ticket: one zero-initialised counter (the kernel leaves it at zero)
cudaError_t launch_cluster(const float *snr_map, const int32_t *argmax, int npix, int nx, float threshold,
                           const float *psf, const uint8_t *mask, int mh, int mw, int topn, void *ws,
                           unsigned int *ticket, nsfrb_cand *top, double *wsnr, int32_t *members, int32_t *result,
                           cudaStream_t st);
// the same kernel with its workspace in a file-scope __device__ array (nsfrb_cluster.cu): allocates nothing
int cluster_static_max_npix();
cudaError_t launch_cluster_static(const float *snr_map, const int32_t *argmax, int npix, int nx, float threshold,
                                  const float *psf, const uint8_t *mask, int mh, int mw, int topn, nsfrb_cand *top,
                                  double *wsnr, int32_t *members, int32_t *result, cudaStream_t st);
size_t search_smem_bytes(int nchan, int RS, int H, int tab_cap);
// on-chip ceilings (nsfrb_peaks.cu)
int peaks_num_tests();
const char *peaks_name(int t);
cudaError_t measure_peaks(int iters, double *per_s, double *per_clk_sm, cudaStream_t st);
size_t final_smem_bytes(int nt);

} // namespace nsfrb
