// Internal declarations shared by nsfrb_api.cu (plan, C ABI) and nsfrb_kernels.cu (sm_100a
// kernels).  Nothing here is part of the public ABI (include/nsfrb.h) and nothing here is
// shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

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

cudaError_t launch_transpose(const float *cube, float *W, int npix, int nchan, int nt, int pitch,
                             cudaStream_t st);
cudaError_t launch_push(const float *chunk, float *W, float *base, int npix, int nchan, int chunk_nt,
                        int pitch, int ring_L, int slot0, int set_base, cudaStream_t st);
cudaError_t launch_search(const SearchParams &p, size_t smem_bytes, cudaStream_t st);
cudaError_t launch_finalize(const FinalParams &p, size_t smem_bytes, cudaStream_t st);
cudaError_t launch_compact(const float *snr_map, const int32_t *argmax, int npix, float threshold,
                           nsfrb_cand *cands, uint32_t cap, uint32_t *ncands, cudaStream_t st);
cudaError_t configure_kernels(size_t final_smem);
cudaError_t configure_search(size_t search_smem);
size_t search_smem_bytes(int nchan, int RS, int H, int tab_cap);
size_t final_smem_bytes(int nt);

} // namespace nsfrb
