// C ABI (include/nsfrb.h) and the host-side plan: validation, delay table (a0), trial
// de-duplication and grouping, workspace, launch sequencing.  All arithmetic of the search
// itself is in nsfrb_kernels.cu.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <numeric>
#include <string>
#include <vector>

#include "nsfrb_internal.h"

using namespace nsfrb;

namespace {

thread_local std::string g_err = "";

int fail(int code, const std::string &msg)
{
    g_err = msg;
    return code;
}
int fail_cuda(cudaError_t e, const char *what)
{
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    cudaGetLastError(); // clear non-sticky error state
    return NSFRB_ECUDA;
}
#define CU(call, what)                                         \
    do {                                                       \
        cudaError_t e__ = (call);                              \
        if (e__ != cudaSuccess) return fail_cuda(e__, what);   \
    } while (0)

inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

constexpr size_t kMaxSmem = 227 * 1024; // opt-in dynamic shared memory per CTA on sm_100

} // namespace

int nsfrb::api_fail(int code, const std::string &msg) { return fail(code, msg); }

void nsfrb::free_plan(nsfrb_plan *p)
{
    if (!p) return;
    cudaFree(p->d_W); cudaFree(p->d_delays_u); cudaFree(p->d_dmax_u); cudaFree(p->d_k_of_u);
    cudaFree(p->d_dd_tab); cudaFree(p->d_dd_off);
    cudaFree(p->d_widths); cudaFree(p->d_j_of_used); cudaFree(p->d_partials); cudaFree(p->d_in); cudaFree(p->d_snr);
    cudaFree(p->d_arg); cudaFree(p->d_cands); cudaFree(p->d_ncands);
    cudaFree(p->d_cluster_ws);
    for (auto &e : p->ev) if (e) cudaEventDestroy(e);
    stream_free(p);
    search4_free(p);
    cudaGetLastError();
    delete p;
}

namespace {

template <typename T>
cudaError_t upload(T **dst, const std::vector<T> &src, size_t *acc)
{
    const size_t bytes = std::max<size_t>(src.size(), 1) * sizeof(T);
    cudaError_t e = cudaMalloc(reinterpret_cast<void **>(dst), bytes);
    if (e != cudaSuccess) return e;
    *acc += bytes;
    if (!src.empty()) e = cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice);
    return e;
}

inline void mark(nsfrb_plan *pl, int i, cudaStream_t st)
{
    if (pl->profiling && pl->ev[i]) cudaEventRecord(pl->ev[i], st);
}

// Dedispersion record streams, one per group of kSearchWarps unique trials (sorted by dmax), read by
// phase 1 of k_search.  All records are 4-int aligned.  Offsets index the raw tile raw[c*RS + i].
//   [0..3]   pos(half 0), pos(half 1), 0, 0
//   half:    {nser, 0, 0, 0} then nser trial records (a half is 8 consecutive trials of the group)
//   trial:   {n, 0, 0, 0} + n offsets c*RS + d[u][c]  (padded to 4 ints): D = sum_c raw[off_c + t]
//        or  {n, 1, 0, 0} + n*4 (new, old) offset pairs: D += sum raw[new + t] - raw[old + t]
//            for the channels whose delay differs from the previous trial (padding pairs are (0,0)).
void build_dd_tables(nsfrb_plan *pl)
{
    const int nchan = pl->nchan, RS = pl->RS;
    pl->dd_tab.clear();
    pl->dd_off.assign(1, 0);
    int cap = 0;
    for (int g = 0; g < pl->n_groups; ++g) {
        std::vector<int32_t> t(4, 0);
        const int u0 = g * kSearchWarps, n = std::min(kSearchWarps, pl->nuniq - u0);
        for (int h = 0; h < 2; ++h) {
            t[h] = (int32_t)t.size();
            const int first = h * 8, nser = std::max(0, std::min(8, n - first));
            t.insert(t.end(), {nser, 0, 0, 0});
            for (int s = 0; s < nser; ++s) {
                const int32_t *d = &pl->delays_u[(size_t)(u0 + first + s) * nchan];
                std::vector<int32_t> pairs;
                if (s > 0) {
                    const int32_t *dp = d - nchan;
                    for (int c = 0; c < nchan; ++c)
                        if (d[c] != dp[c]) { pairs.push_back(c * RS + d[c]); pairs.push_back(c * RS + dp[c]); }
                }
                const int np4 = (int)((pairs.size() / 2 + 3) / 4);
                if (s > 0 && 2 * 4 * np4 < nchan) {
                    pairs.resize((size_t)np4 * 8, 0);
                    t.insert(t.end(), {np4, 1, 0, 0});
                    t.insert(t.end(), pairs.begin(), pairs.end());
                } else {
                    t.insert(t.end(), {nchan, 0, 0, 0});
                    for (int c = 0; c < nchan; ++c) t.push_back(c * RS + d[c]);
                    while (t.size() % 4) t.push_back(0);
                }
            }
        }
        cap = std::max(cap, (int)t.size());
        pl->dd_tab.insert(pl->dd_tab.end(), t.begin(), t.end());
        pl->dd_off.push_back((int32_t)pl->dd_tab.size());
    }
    pl->tab_cap = round_up(std::max(cap, 4), 4);
}

// Generic path (plans k_search4 does not take): search + finalize + compaction over the full-size workspace d_W.
int run_search(nsfrb_plan *pl, int origin, int len, int raw_end_min, int t_offset, cudaStream_t st, float *snr_map,
               int32_t *argmax, nsfrb_cand *cands, uint32_t cap, uint32_t *ncands, int *launches)
{
    const int slices = (pl->nw_used > 0) ? pl->n_groups * pl->n_wb : 0;
    if (slices > 0) {
        SearchParams sp;
        sp.W = pl->d_W; sp.delays_u = pl->d_delays_u; sp.dmax_u = pl->d_dmax_u; sp.k_of_u = pl->d_k_of_u;
        sp.widths = pl->d_widths; sp.partials = pl->d_partials; sp.dd_tab = pl->d_dd_tab; sp.dd_off = pl->d_dd_off;
        sp.npix = pl->npix; sp.nchan = pl->nchan; sp.pitch = pl->pitch; sp.ring_L = pl->nt;
        sp.origin = origin; sp.len = len; sp.raw_end_min = raw_end_min;
        sp.nuniq = pl->nuniq; sp.nw = pl->nw_used; sp.n_groups = pl->n_groups; sp.n_wb = pl->n_wb;
        sp.H = pl->H; sp.RS = pl->RS; sp.wmax = pl->wmax_used; sp.tab_cap = pl->tab_cap;
        CU(launch_search(sp, pl->smem_search, st), "k_search launch");
        ++*launches;
    }
    mark(pl, 2, st);
    FinalParams fp;
    fp.W = pl->d_W; fp.delays_u = pl->d_delays_u; fp.dmax_u = pl->d_dmax_u; fp.widths = pl->d_widths;
    fp.partials = pl->d_partials; fp.snr_map = snr_map; fp.argmax = argmax;
    fp.npix = pl->npix; fp.nchan = pl->nchan; fp.pitch = pl->pitch; fp.ring_L = pl->nt;
    fp.origin = origin; fp.len = len; fp.raw_end_min = raw_end_min; fp.slices = slices; fp.t_offset = t_offset;
    fp.j_of_used = pl->d_j_of_used;
    CU(launch_finalize(fp, pl->smem_final, st), "k_finalize launch");
    ++*launches;
    mark(pl, 3, st);
    CU(cudaMemsetAsync(ncands, 0, sizeof(uint32_t), st), "memset ncands");
    CU(launch_compact(snr_map, argmax, pl->npix, pl->threshold, cands, cap, ncands, st), "k_compact launch");
    ++*launches;
    mark(pl, 4, st);
    pl->ev_valid = pl->profiling;
    return NSFRB_OK;
}

// Calls run on the plan's device whatever device is current in the calling thread; the caller's device is restored.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int dev)
    {
        int cur = -1;
        err = cudaGetDevice(&cur);
        if (err == cudaSuccess && cur != dev) {
            err = cudaSetDevice(dev);
            if (err == cudaSuccess) prev = cur;
        }
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define ON_PLAN_DEVICE(pl)              \
    DeviceGuard guard__((pl)->device);  \
    if (guard__.err != cudaSuccess) return fail_cuda(guard__.err, "cudaSetDevice(plan device)")

// full-size time-contiguous copy of the cube (generic path only), allocated on first use
int ensure_full_workspace(nsfrb_plan *pl)
{
    if (pl->d_W) return NSFRB_OK;
    const size_t wb = (size_t)pl->npix * pl->nchan * (size_t)pl->pitch * sizeof(float);
    cudaError_t e = cudaMalloc(reinterpret_cast<void **>(&pl->d_W), wb);
    if (e == cudaSuccess) e = cudaMemset(pl->d_W, 0, wb);
    if (e != cudaSuccess) {
        cudaFree(pl->d_W);
        pl->d_W = nullptr;
        return e == cudaErrorMemoryAllocation ? fail(NSFRB_ENOMEM, "workspace allocation failed") : fail_cuda(e, "workspace alloc");
    }
    pl->workspace_bytes += wb;
    return NSFRB_OK;
}

int check_outputs(const void *snr_map, const void *argmax, const void *cands, uint32_t cap, const void *ncands)
{
    if (!snr_map || !argmax || !ncands) return fail(NSFRB_EINVAL, "null output pointer");
    if (cap > 0 && !cands) return fail(NSFRB_EINVAL, "cands is null but cand_capacity > 0");
    return NSFRB_OK;
}

int ensure_host_staging(nsfrb_plan *pl, size_t in_bytes, uint32_t cap)
{
    if (in_bytes > 0 && pl->d_in_bytes < in_bytes) {
        cudaFree(pl->d_in); pl->d_in = nullptr; pl->d_in_bytes = 0;
        CU(cudaMalloc(reinterpret_cast<void **>(&pl->d_in), in_bytes), "staging input alloc");
        pl->d_in_bytes = in_bytes;
    }
    if (!pl->d_snr) CU(cudaMalloc(reinterpret_cast<void **>(&pl->d_snr), (size_t)pl->npix * sizeof(float)), "staging snr alloc");
    if (!pl->d_arg) CU(cudaMalloc(reinterpret_cast<void **>(&pl->d_arg), 3 * (size_t)pl->npix * sizeof(int32_t)), "staging argmax alloc");
    if (!pl->d_ncands) CU(cudaMalloc(reinterpret_cast<void **>(&pl->d_ncands), sizeof(uint32_t)), "staging ncands alloc");
    if (cap > pl->d_cands_cap) {
        cudaFree(pl->d_cands); pl->d_cands = nullptr; pl->d_cands_cap = 0;
        CU(cudaMalloc(reinterpret_cast<void **>(&pl->d_cands), (size_t)cap * sizeof(nsfrb_cand)), "staging cands alloc");
        pl->d_cands_cap = cap;
    }
    return NSFRB_OK;
}

int copy_back(nsfrb_plan *pl, cudaStream_t st, float *snr_h, int32_t *arg_h, nsfrb_cand *cands_h, uint32_t cap,
              uint32_t *ncands_h)
{
    CU(cudaMemcpyAsync(snr_h, pl->d_snr, (size_t)pl->npix * sizeof(float), cudaMemcpyDeviceToHost, st), "D2H snr");
    CU(cudaMemcpyAsync(arg_h, pl->d_arg, 3 * (size_t)pl->npix * sizeof(int32_t), cudaMemcpyDeviceToHost, st), "D2H argmax");
    CU(cudaMemcpyAsync(ncands_h, pl->d_ncands, sizeof(uint32_t), cudaMemcpyDeviceToHost, st), "D2H ncands");
    CU(cudaStreamSynchronize(st), "stream sync");
    const uint32_t n = std::min(*ncands_h, cap);
    if (n > 0) {
        CU(cudaMemcpyAsync(cands_h, pl->d_cands, (size_t)n * sizeof(nsfrb_cand), cudaMemcpyDeviceToHost, st), "D2H cands");
        CU(cudaStreamSynchronize(st), "stream sync");
    }
    return NSFRB_OK;
}

void pipe_free(nsfrb_plan *pl)
{
    auto *pp = pl->pipe;
    if (!pp) return;
    for (int b = 0; b < 2; ++b) {
        if (pp->done[b]) cudaEventSynchronize(pp->done[b]);
        cudaFree(pp->d_in[b]); cudaFree(pp->d_snr[b]); cudaFree(pp->d_arg[b]); cudaFree(pp->d_cands[b]);
        cudaFree(pp->d_ncands[b]);
        if (pp->copied[b]) cudaEventDestroy(pp->copied[b]);
        if (pp->done[b]) cudaEventDestroy(pp->done[b]);
    }
    if (pp->s_copy) cudaStreamDestroy(pp->s_copy);
    if (pp->s_comp) cudaStreamDestroy(pp->s_comp);
    delete pp;
    pl->pipe = nullptr;
}

int pipe_slot(nsfrb_plan *pl, int b, size_t in_bytes, uint32_t cap)
{
    if (!pl->pipe) {
        pl->pipe = new (std::nothrow) nsfrb_plan::HostPipe();
        if (!pl->pipe) return fail(NSFRB_ENOMEM, "out of host memory");
        CU(cudaStreamCreateWithFlags(&pl->pipe->s_copy, cudaStreamNonBlocking), "copy stream");
        CU(cudaStreamCreateWithFlags(&pl->pipe->s_comp, cudaStreamNonBlocking), "compute stream");
    }
    auto *pp = pl->pipe;
    if (!pp->copied[b]) CU(cudaEventCreateWithFlags(&pp->copied[b], cudaEventDisableTiming), "event");
    if (!pp->done[b]) CU(cudaEventCreateWithFlags(&pp->done[b], cudaEventDisableTiming), "event");
    if (pp->busy[b]) {   // the push that used this slot two calls ago: its staging and host outputs must be complete
        CU(cudaEventSynchronize(pp->done[b]), "wait for the slot");
        pp->busy[b] = false;
    }
    if (pp->in_bytes[b] < in_bytes) {
        cudaFree(pp->d_in[b]); pp->d_in[b] = nullptr; pp->in_bytes[b] = 0;
        CU(cudaMalloc(reinterpret_cast<void **>(&pp->d_in[b]), in_bytes), "staging input alloc");
        pp->in_bytes[b] = in_bytes;
    }
    if (!pp->d_snr[b]) CU(cudaMalloc(reinterpret_cast<void **>(&pp->d_snr[b]), (size_t)pl->npix * sizeof(float)), "staging alloc");
    if (!pp->d_arg[b]) CU(cudaMalloc(reinterpret_cast<void **>(&pp->d_arg[b]), 3 * (size_t)pl->npix * sizeof(int32_t)), "staging alloc");
    if (!pp->d_ncands[b]) CU(cudaMalloc(reinterpret_cast<void **>(&pp->d_ncands[b]), sizeof(uint32_t)), "staging alloc");
    if (cap > pp->cands_cap[b]) {
        cudaFree(pp->d_cands[b]); pp->d_cands[b] = nullptr; pp->cands_cap[b] = 0;
        CU(cudaMalloc(reinterpret_cast<void **>(&pp->d_cands[b]), (size_t)cap * sizeof(nsfrb_cand)), "staging alloc");
        pp->cands_cap[b] = cap;
    }
    return NSFRB_OK;
}

} // namespace

#pragma GCC visibility push(default)
extern "C" {

const char *nsfrb_last_error(void) { return g_err.c_str(); }
const char *nsfrb_version(void) { return "0.1 (sm_100a)"; }

} // extern "C"
#pragma GCC visibility pop

// Validation and every host-side table of a plan (no CUDA call): shared by nsfrb_plan_create and the
// JIT harness entry points, which must work on a machine without a GPU.
int nsfrb::plan_host_init(nsfrb_plan **out, int nx, int ny, int nchan, int nt, const double *freqs_GHz, double tsamp_s,
                          const double *dm_list, int ndm, const int32_t *width_list, int nwidth, float threshold)
{
    if (!out) return fail(NSFRB_EINVAL, "out is null");
    *out = nullptr;
    if (!freqs_GHz || !dm_list || !width_list) return fail(NSFRB_EINVAL, "null input list");
    if (nx < 1 || ny < 1 || nchan < 1 || nt < 1 || ndm < 1 || nwidth < 1) return fail(NSFRB_EINVAL, "non-positive size");
    if ((long long)nx * ny > 0x7fffffffLL / 4) return fail(NSFRB_EINVAL, "image too large");
    if (!(tsamp_s > 0.0) || !std::isfinite(tsamp_s)) return fail(NSFRB_EINVAL, "tsamp_s must be finite and > 0");
    if (!std::isfinite(threshold) && !(threshold == INFINITY || threshold == -INFINITY))
        return fail(NSFRB_EINVAL, "threshold is NaN");
    for (int c = 0; c < nchan; ++c)
        if (!std::isfinite(freqs_GHz[c]) || !(freqs_GHz[c] > 0.0)) return fail(NSFRB_EINVAL, "freqs_GHz must be finite and > 0");
    for (int k = 0; k < ndm; ++k)
        if (!std::isfinite(dm_list[k]) || dm_list[k] < 0.0) return fail(NSFRB_EINVAL, "dm_list must be finite and >= 0");
    for (int j = 0; j < nwidth; ++j) {
        if (width_list[j] < 1) return fail(NSFRB_EINVAL, "width < 1");
        for (int i = 0; i < j; ++i)
            if (width_list[i] == width_list[j]) return fail(NSFRB_EINVAL, "duplicate width");
    }

    nsfrb_plan *pl = new (std::nothrow) nsfrb_plan();
    if (!pl) return fail(NSFRB_ENOMEM, "host allocation failed");
    pl->nx = nx; pl->ny = ny; pl->npix = nx * ny; pl->nchan = nchan; pl->nt = nt; pl->ndm = ndm; pl->nw = nwidth;
    pl->tsamp = tsamp_s; pl->threshold = threshold;
    pl->freqs.assign(freqs_GHz, freqs_GHz + nchan);
    pl->dms.assign(dm_list, dm_list + ndm);
    pl->widths.assign(width_list, width_list + nwidth);

    // ---- a0: delay table, float64 on the host (include/nsfrb.h formula)
    double f_ref = freqs_GHz[0];
    for (int c = 1; c < nchan; ++c) f_ref = std::max(f_ref, freqs_GHz[c]);
    const double inv_ref2 = 1.0 / (f_ref * f_ref);
    pl->delays.resize((size_t)ndm * nchan);
    pl->dmax.resize(ndm);
    for (int k = 0; k < ndm; ++k) {
        const double scale = 4.15e-3 * dm_list[k];
        int mx = 0;
        for (int c = 0; c < nchan; ++c) {
            const double inv2 = 1.0 / (freqs_GHz[c] * freqs_GHz[c]);
            const double x = (scale * (inv2 - inv_ref2)) / tsamp_s;
            const double r = std::floor(x + 0.5);
            if (!(r < (double)nt)) {
                free_plan(pl);
                return fail(NSFRB_EINVAL, "a trial's delay reaches nt: no valid sample left (nt <= dmax_k)");
            }
            const int d = (int)r;
            pl->delays[(size_t)k * nchan + c] = d;
            mx = std::max(mx, d);
        }
        pl->dmax[k] = mx;
    }

    // ---- unique delay vectors (a duplicate can never win under the lowest-index tie-break)
    std::vector<int> first;
    for (int k = 0; k < ndm; ++k) {
        bool dup = false;
        for (int u : first)
            if (std::memcmp(&pl->delays[(size_t)u * nchan], &pl->delays[(size_t)k * nchan], sizeof(int32_t) * nchan) == 0) {
                dup = true;
                break;
            }
        if (!dup) first.push_back(k);
    }
    std::stable_sort(first.begin(), first.end(), [&](int a, int b) { return pl->dmax[a] < pl->dmax[b]; });
    pl->nuniq = (int)first.size();
    for (int k : first) {
        pl->k_of_u.push_back(k);
        pl->dmax_u.push_back(pl->dmax[k]);
        pl->delays_u.insert(pl->delays_u.end(), pl->delays.begin() + (size_t)k * nchan,
                            pl->delays.begin() + (size_t)(k + 1) * nchan);
    }
    pl->dmax_all = *std::max_element(pl->dmax.begin(), pl->dmax.end());
    pl->dmin_all = *std::min_element(pl->dmax.begin(), pl->dmax.end());

    // ---- widths that can hold a cell for at least one trial
    const int T_longest = nt - pl->dmin_all;
    for (int j = 0; j < nwidth; ++j)
        if (width_list[j] <= T_longest) {
            pl->widths_used.push_back(width_list[j]);
            pl->j_of_used.push_back(j);
            pl->wmax_used = std::max(pl->wmax_used, width_list[j]);
        }
    pl->nw_used = (int)pl->widths_used.size();
    pl->stream_worder.resize(pl->nw_used);
    std::iota(pl->stream_worder.begin(), pl->stream_worder.end(), 0);
    std::sort(pl->stream_worder.begin(), pl->stream_worder.end(),
              [&](int a, int b) { return pl->widths_used[a] < pl->widths_used[b]; });

    for (int k = 0; k < ndm; ++k) {
        const int T = nt - pl->dmax[k];
        pl->shift_adds_per_pixel += (int64_t)nchan * T;
        for (int j = 0; j < nwidth; ++j)
            if (T - width_list[j] + 1 > 0) pl->cells_per_pixel += T - width_list[j] + 1;
    }

    // ---- kernel geometry
    pl->n_groups = (pl->nuniq + kSearchWarps - 1) / kSearchWarps;
    pl->n_wb = std::max(1, (pl->nw_used + kWidthBatch - 1) / kWidthBatch);
    pl->H = round_up(std::max(pl->wmax_used, 1) + kBlockLen + 32, 32);
    {   // a power-of-two ring makes every wrap one AND (generic k_search); take it when the shared memory allows
        int h2 = 32;
        while (h2 < pl->H) h2 <<= 1;
        const int RS0 = round_up(kBlockLen + pl->dmax_all, 4);
        if (search_smem_bytes(nchan, RS0, h2, 4096) + 4096 <= kMaxSmem) pl->H = h2;
    }
    pl->RS = round_up(kBlockLen + pl->dmax_all, 4);
    pl->pitch = round_up(nt, 4);
    build_dd_tables(pl);
    pl->smem_search = search_smem_bytes(nchan, pl->RS, pl->H, pl->tab_cap);
    pl->smem_final = final_smem_bytes(nt);
    if (pl->smem_search > kMaxSmem || pl->smem_final > kMaxSmem) {
        char buf[256];
        snprintf(buf, sizeof buf,
                 "problem does not fit shared memory: search needs %zu B (nchan*%d + %d*%d floats), finalize %zu B; limit %zu B",
                 pl->smem_search, pl->RS, kSearchWarps, pl->H, pl->smem_final, kMaxSmem);
        free_plan(pl);
        return fail(NSFRB_ENOMEM, buf);
    }
    if ((long long)pl->npix * pl->n_groups * pl->n_wb > 0x7fffffffLL) {
        free_plan(pl);
        return fail(NSFRB_EINVAL, "too many (pixel, DM group, width batch) tasks for one launch");
    }

    *out = pl;
    return NSFRB_OK;
}

#pragma GCC visibility push(default)
extern "C" {

int nsfrb_plan_create(nsfrb_plan **out, int nx, int ny, int nchan, int nt, const double *freqs_GHz, double tsamp_s,
                      const double *dm_list, int ndm, const int32_t *width_list, int nwidth, float threshold)
{
    nsfrb_plan *pl = nullptr;
    if (int rc = plan_host_init(&pl, nx, ny, nchan, nt, freqs_GHz, tsamp_s, dm_list, ndm, width_list, nwidth, threshold))
        return rc;
    *out = nullptr;
    // ---- device state
    cudaError_t e = cudaGetDevice(&pl->device);
    size_t acc = 0;
    if (e == cudaSuccess) e = upload(&pl->d_delays_u, pl->delays_u, &acc);
    if (e == cudaSuccess) e = upload(&pl->d_dd_tab, pl->dd_tab, &acc);
    if (e == cudaSuccess) e = upload(&pl->d_dd_off, pl->dd_off, &acc);
    if (e == cudaSuccess) e = upload(&pl->d_dmax_u, pl->dmax_u, &acc);
    if (e == cudaSuccess) e = upload(&pl->d_k_of_u, pl->k_of_u, &acc);
    if (e == cudaSuccess) e = upload(&pl->d_widths, pl->widths_used, &acc);
    if (e == cudaSuccess) e = upload(&pl->d_j_of_used, pl->j_of_used, &acc);
    if (e == cudaSuccess) {
        const size_t pb = (size_t)pl->npix * std::max(pl->n_groups * pl->n_wb, (pl->nuniq + 7) / 8) * sizeof(Partial);
        e = cudaMalloc(reinterpret_cast<void **>(&pl->d_partials), pb);
        acc += pb;
    }
    if (e != cudaSuccess) {
        const int code = (e == cudaErrorMemoryAllocation) ? NSFRB_ENOMEM : NSFRB_ECUDA;
        std::string msg = std::string("plan device setup: ") + cudaGetErrorString(e);
        cudaGetLastError();
        free_plan(pl);
        return fail(code, msg);
    }
    pl->workspace_bytes = acc;
    *out = pl;
    return NSFRB_OK;
}

int nsfrb_plan_prepare(nsfrb_plan *pl, int mode, int chunk_nt)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    ON_PLAN_DEVICE(pl);
    std::string err;
    if (mode == NSFRB_PREPARE_SEARCH) {
        if (search4_usable(pl)) {
            if (int rc = search4_prepare(pl, err)) return fail(rc, err);
            return NSFRB_OK;
        }
        return ensure_full_workspace(pl);
    }
    if (mode == NSFRB_PREPARE_STREAM) {
        if (chunk_nt < 1 || chunk_nt > pl->nt) return fail(NSFRB_EINVAL, "chunk_nt must be in [1, nt]");
        if (int rc = stream_prepare(pl, chunk_nt, err)) return fail(rc, err);
        return NSFRB_OK;
    }
    return fail(NSFRB_EINVAL, "mode must be NSFRB_PREPARE_SEARCH or NSFRB_PREPARE_STREAM");
}

int nsfrb_search(nsfrb_plan *pl, const float *cube, void *stream, float *snr_map, int32_t *argmax, nsfrb_cand *cands,
                 uint32_t cand_capacity, uint32_t *ncands)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    if (!cube) return fail(NSFRB_EINVAL, "cube is null");
    if ((reinterpret_cast<uintptr_t>(cube) & 15u) != 0) return fail(NSFRB_EINVAL, "cube is not 16-byte aligned");
    if (int rc = check_outputs(snr_map, argmax, cands, cand_capacity, ncands)) return rc;
    if (pl->n_received != 0) return fail(NSFRB_ESTATE, "plan holds streamed samples; call nsfrb_stream_reset first");
    ON_PLAN_DEVICE(pl);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int launches = 0;
    if (search4_usable(pl)) { // plan-specialised kernel over pixel batches; it also writes snr_map/argmax (a6)
        mark(pl, 0, st);
        std::string err;
        if (int rc = search4_launch(pl, cube, st, snr_map, argmax, &launches, (pl->profiling && pl->ev[1]) ? pl->ev[1] : nullptr, err))
            return fail(rc, err);
        mark(pl, 2, st);
        mark(pl, 3, st);
        CU(cudaMemsetAsync(ncands, 0, sizeof(uint32_t), st), "memset ncands");
        CU(launch_compact(snr_map, argmax, pl->npix, pl->threshold, cands, cand_capacity, ncands, st), "k_compact launch");
        ++launches;
        mark(pl, 4, st);
        pl->ev_valid = pl->profiling;
        pl->last_launches = launches;
        return NSFRB_OK;
    }
    if (int rc = ensure_full_workspace(pl)) return rc;
    mark(pl, 0, st);
    CU(launch_transpose(cube, pl->d_W, pl->npix, pl->nchan, pl->nt, pl->pitch, 0, pl->npix, st), "k_transpose launch");
    ++launches;
    mark(pl, 1, st);
    const int rc = run_search(pl, 0, pl->nt, 0, 0, st, snr_map, argmax, cands, cand_capacity, ncands, &launches);
    pl->last_launches = launches;
    return rc;
}

int nsfrb_stream_push(nsfrb_plan *pl, const float *chunk, int chunk_nt, void *stream, float *snr_map, int32_t *argmax,
                      nsfrb_cand *cands, uint32_t cand_capacity, uint32_t *ncands)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    if (!chunk) return fail(NSFRB_EINVAL, "chunk is null");
    if ((reinterpret_cast<uintptr_t>(chunk) & 15u) != 0) return fail(NSFRB_EINVAL, "chunk is not 16-byte aligned");
    if (chunk_nt < 1 || chunk_nt > pl->nt) return fail(NSFRB_EINVAL, "chunk_nt must be in [1, nt]");
    if (int rc = check_outputs(snr_map, argmax, cands, cand_capacity, ncands)) return rc;
    ON_PLAN_DEVICE(pl);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int launches = 0;
    mark(pl, 0, st);
    std::string err;
    if (int rc = stream_push(pl, chunk, chunk_nt, st, snr_map, argmax, &launches, err)) return fail(rc, err);
    mark(pl, 3, st);
    CU(cudaMemsetAsync(ncands, 0, sizeof(uint32_t), st), "memset ncands");
    CU(launch_compact(snr_map, argmax, pl->npix, pl->threshold, cands, cand_capacity, ncands, st), "k_compact launch");
    ++launches;
    mark(pl, 4, st);
    pl->ev_valid = pl->profiling;
    pl->last_launches = launches;
    return NSFRB_OK;
}

int nsfrb_stream_set_cubes(nsfrb_plan *pl, float *snr_cube, int32_t *toa_cube)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    std::string err;
    if (int rc = stream_set_cubes(pl, snr_cube, toa_cube, err)) return fail(rc, err);
    return NSFRB_OK;
}

int nsfrb_stream_set_running_sigma(nsfrb_plan *pl, double alpha, float *snr_map_run, int32_t *argmax_run)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    std::string err;
    if (int rc = stream_set_running(pl, alpha, snr_map_run, argmax_run, err)) return fail(rc, err);
    return NSFRB_OK;
}

int nsfrb_stream_reset(nsfrb_plan *pl)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    if (pl->pipe)   // pipelined pushes still in flight read and write the ring
        for (int b = 0; b < 2; ++b)
            if (pl->pipe->busy[b]) {
                CU(cudaEventSynchronize(pl->pipe->done[b]), "wait");
                pl->pipe->busy[b] = false;
            }
    pl->n_received = 0;
    stream_reset(pl);
    return NSFRB_OK;
}

int nsfrb_search_host(nsfrb_plan *pl, const float *cube_host, void *stream, float *snr_map_host, int32_t *argmax_host,
                      nsfrb_cand *cands_host, uint32_t cand_capacity, uint32_t *ncands_host)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    if (!cube_host) return fail(NSFRB_EINVAL, "cube is null");
    if (int rc = check_outputs(snr_map_host, argmax_host, cands_host, cand_capacity, ncands_host)) return rc;
    if (pl->n_received != 0) return fail(NSFRB_ESTATE, "plan holds streamed samples; call nsfrb_stream_reset first");
    ON_PLAN_DEVICE(pl);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (search4_usable(pl)) {
        // pixel batches straight from the host cube: no cube-sized staging buffer, copies overlap the search
        if (int rc = ensure_host_staging(pl, 0, cand_capacity)) return rc;
        int launches = 0;
        std::string err;
        if (int rc = search4_launch_host(pl, cube_host, st, pl->d_snr, pl->d_arg, &launches, err)) return fail(rc, err);
        CU(cudaMemsetAsync(pl->d_ncands, 0, sizeof(uint32_t), st), "memset ncands");
        CU(launch_compact(pl->d_snr, pl->d_arg, pl->npix, pl->threshold, pl->d_cands, cand_capacity, pl->d_ncands, st), "k_compact launch");
        pl->last_launches = launches + 1;
        return copy_back(pl, st, snr_map_host, argmax_host, cands_host, cand_capacity, ncands_host);
    }
    const size_t bytes = (size_t)pl->nchan * pl->nt * (size_t)pl->npix * sizeof(float);
    if (int rc = ensure_host_staging(pl, bytes, cand_capacity)) return rc;
    CU(cudaMemcpyAsync(pl->d_in, cube_host, bytes, cudaMemcpyHostToDevice, st), "H2D cube");
    if (int rc = nsfrb_search(pl, pl->d_in, stream, pl->d_snr, pl->d_arg, pl->d_cands, cand_capacity, pl->d_ncands)) return rc;
    return copy_back(pl, st, snr_map_host, argmax_host, cands_host, cand_capacity, ncands_host);
}

int nsfrb_stream_push_host(nsfrb_plan *pl, const float *chunk_host, int chunk_nt, void *stream, float *snr_map_host,
                           int32_t *argmax_host, nsfrb_cand *cands_host, uint32_t cand_capacity, uint32_t *ncands_host)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    if (!chunk_host) return fail(NSFRB_EINVAL, "chunk is null");
    if (chunk_nt < 1 || chunk_nt > pl->nt) return fail(NSFRB_EINVAL, "chunk_nt must be in [1, nt]");
    if (int rc = check_outputs(snr_map_host, argmax_host, cands_host, cand_capacity, ncands_host)) return rc;
    ON_PLAN_DEVICE(pl);
    const size_t bytes = (size_t)pl->nchan * chunk_nt * (size_t)pl->npix * sizeof(float);
    if (int rc = ensure_host_staging(pl, bytes, cand_capacity)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    CU(cudaMemcpyAsync(pl->d_in, chunk_host, bytes, cudaMemcpyHostToDevice, st), "H2D chunk");
    if (int rc = nsfrb_stream_push(pl, pl->d_in, chunk_nt, stream, pl->d_snr, pl->d_arg, pl->d_cands, cand_capacity,
                                   pl->d_ncands))
        return rc;
    return copy_back(pl, st, snr_map_host, argmax_host, cands_host, cand_capacity, ncands_host);
}

int nsfrb_stream_push_host_async(nsfrb_plan *pl, const float *chunk_host, int chunk_nt, float *snr_map_host,
                                 int32_t *argmax_host, nsfrb_cand *cands_host, uint32_t cand_capacity,
                                 uint32_t *ncands_host)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    if (!chunk_host) return fail(NSFRB_EINVAL, "chunk is null");
    if (chunk_nt < 1 || chunk_nt > pl->nt) return fail(NSFRB_EINVAL, "chunk_nt must be in [1, nt]");
    if (int rc = check_outputs(snr_map_host, argmax_host, cands_host, cand_capacity, ncands_host)) return rc;
    ON_PLAN_DEVICE(pl);
    const size_t bytes = (size_t)pl->nchan * chunk_nt * (size_t)pl->npix * sizeof(float);
    const int b = pl->pipe ? (int)(pl->pipe->count & 1) : 0;
    if (int rc = pipe_slot(pl, b, bytes, cand_capacity)) return rc;
    auto *pp = pl->pipe;
    // copy stream: chunk i+1 travels while the compute stream still works on chunk i
    CU(cudaMemcpyAsync(pp->d_in[b], chunk_host, bytes, cudaMemcpyHostToDevice, pp->s_copy), "H2D chunk");
    CU(cudaEventRecord(pp->copied[b], pp->s_copy), "event record");
    CU(cudaStreamWaitEvent(pp->s_comp, pp->copied[b], 0), "stream wait");
    if (int rc = nsfrb_stream_push(pl, pp->d_in[b], chunk_nt, pp->s_comp, pp->d_snr[b], pp->d_arg[b], pp->d_cands[b],
                                   cand_capacity, pp->d_ncands[b]))
        return rc;
    CU(cudaMemcpyAsync(snr_map_host, pp->d_snr[b], (size_t)pl->npix * sizeof(float), cudaMemcpyDeviceToHost, pp->s_comp), "D2H snr");
    CU(cudaMemcpyAsync(argmax_host, pp->d_arg[b], 3 * (size_t)pl->npix * sizeof(int32_t), cudaMemcpyDeviceToHost, pp->s_comp), "D2H argmax");
    CU(cudaMemcpyAsync(ncands_host, pp->d_ncands[b], sizeof(uint32_t), cudaMemcpyDeviceToHost, pp->s_comp), "D2H ncands");
    if (cand_capacity > 0)   // the count is not known on the host yet: all cand_capacity records travel
        CU(cudaMemcpyAsync(cands_host, pp->d_cands[b], (size_t)cand_capacity * sizeof(nsfrb_cand), cudaMemcpyDeviceToHost, pp->s_comp), "D2H cands");
    CU(cudaEventRecord(pp->done[b], pp->s_comp), "event record");
    pp->busy[b] = true;
    ++pp->count;
    return NSFRB_OK;
}

int nsfrb_stream_wait(nsfrb_plan *pl)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    if (!pl->pipe) return NSFRB_OK;
    for (int b = 0; b < 2; ++b)
        if (pl->pipe->busy[b]) {
            CU(cudaEventSynchronize(pl->pipe->done[b]), "wait");
            pl->pipe->busy[b] = false;
        }
    return NSFRB_OK;
}

int nsfrb_plan_destroy(nsfrb_plan *pl)
{
    if (!pl) return NSFRB_OK;
    cudaDeviceSynchronize();
    pipe_free(pl);
    free_plan(pl);
    return NSFRB_OK;
}

int nsfrb_plan_get_delays(const nsfrb_plan *pl, int32_t *out)
{
    if (!pl || !out) return fail(NSFRB_EINVAL, "null argument");
    std::memcpy(out, pl->delays.data(), pl->delays.size() * sizeof(int32_t));
    return NSFRB_OK;
}

int nsfrb_plan_get_info(const nsfrb_plan *pl, nsfrb_plan_info *info)
{
    if (!pl || !info) return fail(NSFRB_EINVAL, "null argument");
    info->npix = pl->npix; info->nchan = pl->nchan; info->nt = pl->nt; info->ndm = pl->ndm; info->nwidth = pl->nw;
    info->ndm_unique = pl->nuniq; info->dmax = pl->dmax_all; info->wmax = pl->wmax_used;
    info->n_groups = pl->n_groups; info->n_width_batches = pl->n_wb; info->series_per_cta = kSearchWarps;
    info->block_len = kBlockLen; info->ring_len = search4_usable(pl) ? search4_ring_len(pl) : pl->H; info->search_threads = kSearchWarps * 32;
    info->search_smem_bytes = (int64_t)pl->smem_search; info->workspace_bytes = (int64_t)(pl->workspace_bytes + stream_bytes(pl) + search4_bytes(pl));
    info->cells_per_pixel = pl->cells_per_pixel; info->shift_adds_per_pixel = pl->shift_adds_per_pixel;
    return NSFRB_OK;
}

int nsfrb_jit_stream_kernel(int nx, int ny, int nchan, int nt, const double *freqs_GHz, double tsamp_s, const double *dm_list,
                            int ndm, const int32_t *width_list, int nwidth, int chunk_nt, const char *variant, int want_cubin,
                            char *out, size_t capacity, size_t *needed)
{
    if (!needed) return fail(NSFRB_EINVAL, "needed is null");
    nsfrb_plan *pl = nullptr;
    if (int rc = plan_host_init(&pl, nx, ny, nchan, nt, freqs_GHz, tsamp_s, dm_list, ndm, width_list, nwidth, 0.f)) return rc;
    std::string src, err;
    int rc = stream_source(pl, chunk_nt, variant, src, err);
    free_plan(pl);
    if (rc) return fail(rc, err);
    std::vector<char> bin;
    const char *data = src.data();
    size_t n = src.size();
    if (want_cubin) {
        std::string log;
        if ((rc = stream_compile(src, bin, log))) return fail(rc, log);
        data = bin.data();
        n = bin.size();
    }
    *needed = n;
    if (out && capacity >= n) std::memcpy(out, data, n);
    return NSFRB_OK;
}

int nsfrb_jit_search_kernel(int nx, int ny, int nchan, int nt, const double *freqs_GHz, double tsamp_s, const double *dm_list,
                            int ndm, const int32_t *width_list, int nwidth, int want_cubin, char *out, size_t capacity,
                            size_t *needed)
{
    if (!needed) return fail(NSFRB_EINVAL, "needed is null");
    nsfrb_plan *pl = nullptr;
    if (int rc = plan_host_init(&pl, nx, ny, nchan, nt, freqs_GHz, tsamp_s, dm_list, ndm, width_list, nwidth, 0.f)) return rc;
    std::string src, err;
    int rc = search4_source(pl, src, err);
    free_plan(pl);
    if (rc) return fail(rc, err);
    std::vector<char> bin;
    const char *data = src.data();
    size_t n = src.size();
    if (want_cubin) {
        std::string log;
        if ((rc = stream_compile(src, bin, log))) return fail(rc, log);
        data = bin.data();
        n = bin.size();
    }
    *needed = n;
    if (out && capacity >= n) std::memcpy(out, data, n);
    return NSFRB_OK;
}

int nsfrb_bin_time(const float *cube, int nchan, int nt, int64_t npix, int factor, float *out, void *stream)
{
    if (!cube || !out) return fail(NSFRB_EINVAL, "null pointer");
    if (nchan < 1 || nt < 1 || npix < 1 || factor < 1) return fail(NSFRB_EINVAL, "non-positive size or factor");
    if (nchan > 65535) return fail(NSFRB_EINVAL, "too many channels");
    if (cube == out) return fail(NSFRB_EINVAL, "in-place binning is not supported");
    CU(launch_bin(cube, out, nchan, nt, (long long)npix, factor, static_cast<cudaStream_t>(stream)), "k_bin launch");
    return NSFRB_OK;
}

int nsfrb_median_subtract(const float *cube, int nchan, int nt, int64_t npix, float *out, float *median, void *stream)
{
    if (!cube || !out) return fail(NSFRB_EINVAL, "null pointer");
    if (nchan < 1 || nt < 1 || npix < 1) return fail(NSFRB_EINVAL, "non-positive size");
    if (nchan > 65535) return fail(NSFRB_EINVAL, "too many channels");
    if (nt > median_max_nt()) return fail(NSFRB_EINVAL, "nt too large (max 65535)");
    if ((long long)nchan * npix > 0x7fffffffLL * 256) return fail(NSFRB_EINVAL, "too many series");
    CU(launch_median(cube, out, median, nchan, nt, (long long)npix, static_cast<cudaStream_t>(stream)),
       "k_median launch");
    return NSFRB_OK;
}

int nsfrb_psf_mask(const float *psf, int mh, int mw, double percentile, uint8_t *mask, double *value, void *stream)
{
    if (!psf || !mask) return fail(NSFRB_EINVAL, "null pointer");
    if (mh < 1 || mw < 1) return fail(NSFRB_EINVAL, "non-positive PSF size");
    if (!(percentile >= 0.0 && percentile <= 100.0)) return fail(NSFRB_EINVAL, "percentile outside [0, 100]");
    const long long n = (long long)mh * mw;
    if (n > 0x7fffffffLL) return fail(NSFRB_EINVAL, "PSF too large");
    // reading R25: rank q/100*(n-1), linear interpolation between the neighbouring order statistics
    const double r = percentile / 100.0 * (double)(n - 1);
    long long lo = (long long)std::floor(r);
    lo = std::min(std::max(lo, 0LL), n - 1);
    CU(launch_psf_mask(psf, n, lo, r - (double)lo, mask, value, static_cast<cudaStream_t>(stream)), "k_psf_mask launch");
    return NSFRB_OK;
}

int nsfrb_cluster(nsfrb_plan *pl, const float *snr_map, const int32_t *argmax, const float *psf, const uint8_t *mask,
                  int mh, int mw, int topn, nsfrb_cand *top, double *wsnr, int32_t *members, int32_t *result,
                  void *stream)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    if (!snr_map || !argmax || !psf || !mask || !top || !wsnr || !members || !result)
        return fail(NSFRB_EINVAL, "null pointer");
    if (mh < 1 || mw < 1) return fail(NSFRB_EINVAL, "non-positive PSF size");
    if (topn < 1 || topn > cluster_max_top()) return fail(NSFRB_EINVAL, "topn outside 1..32");
    ON_PLAN_DEVICE(pl);
    if (!pl->d_cluster_ws) {
        const size_t bytes = 256 + (size_t)cluster_grid(pl->npix) * cluster_max_top() * sizeof(unsigned long long);
        CU(cudaMalloc(&pl->d_cluster_ws, bytes), "cluster workspace");
        CU(cudaMemset(pl->d_cluster_ws, 0, 256), "cluster workspace");
        pl->workspace_bytes += bytes;
    }
    char *ws = static_cast<char *>(pl->d_cluster_ws);
    CU(launch_cluster(snr_map, argmax, pl->npix, pl->nx, pl->threshold, psf, mask, mh, mw, topn, ws + 256,
                      reinterpret_cast<unsigned int *>(ws), top, wsnr, members, result,
                      static_cast<cudaStream_t>(stream)),
       "k_cluster launch");
    pl->last_launches = 1;
    return NSFRB_OK;
}

int nsfrb_cluster_static(int nx, int ny, float threshold, const float *snr_map, const int32_t *argmax, const float *psf,
                         const uint8_t *mask, int mh, int mw, int topn, nsfrb_cand *top, double *wsnr, int32_t *members,
                         int32_t *result, void *stream)
{
    if (!snr_map || !argmax || !psf || !mask || !top || !wsnr || !members || !result)
        return fail(NSFRB_EINVAL, "null pointer");
    if (nx < 1 || ny < 1) return fail(NSFRB_EINVAL, "non-positive image size");
    if ((long long)nx * ny > (long long)cluster_static_max_npix()) {
        char buf[160];
        snprintf(buf, sizeof buf, "nsfrb_cluster_static: %lld pixels exceed the static workspace's limit of %d (use nsfrb_cluster)",
                 (long long)nx * ny, cluster_static_max_npix());
        return fail(NSFRB_EINVAL, buf);
    }
    if (mh < 1 || mw < 1) return fail(NSFRB_EINVAL, "non-positive PSF size");
    if (topn < 1 || topn > cluster_max_top()) return fail(NSFRB_EINVAL, "topn outside 1..32 (the static workspace holds 32 keys per CTA)");
    if (std::isnan(threshold)) return fail(NSFRB_EINVAL, "threshold is NaN");
    CU(launch_cluster_static(snr_map, argmax, nx * ny, nx, threshold, psf, mask, mh, mw, topn, top, wsnr, members, result,
                             static_cast<cudaStream_t>(stream)),
       "k_cluster launch (static workspace)");
    return NSFRB_OK;
}

int nsfrb_peaks_count(void) { return peaks_num_tests(); }
const char *nsfrb_peaks_name(int test) { return peaks_name(test); }
int nsfrb_measure_peaks(int iters, double *per_s, double *per_clk_sm, void *stream)
{
    if (!per_s || !per_clk_sm) return fail(NSFRB_EINVAL, "null pointer");
    if (iters < 1) return fail(NSFRB_EINVAL, "iters < 1");
    CU(measure_peaks(iters, per_s, per_clk_sm, static_cast<cudaStream_t>(stream)), "peak microbenchmarks");
    return NSFRB_OK;
}

int nsfrb_plan_last_launches(const nsfrb_plan *pl) { return pl ? pl->last_launches : 0; }

int nsfrb_stream_mode(const nsfrb_plan *pl) { return pl ? stream_mode(pl) : 0; }

int nsfrb_plan_set_profiling(nsfrb_plan *pl, int on)
{
    if (!pl) return fail(NSFRB_EINVAL, "plan is null");
    if (on)
        for (auto &e : pl->ev)
            if (!e) CU(cudaEventCreate(&e), "event create");
    pl->profiling = on != 0;
    pl->ev_valid = false;
    return NSFRB_OK;
}

int nsfrb_plan_get_kernel_ms(nsfrb_plan *pl, float out[4])
{
    if (!pl || !out) return fail(NSFRB_EINVAL, "null argument");
    if (!pl->ev_valid) return fail(NSFRB_ESTATE, "no profiled call yet (nsfrb_plan_set_profiling)");
    CU(cudaEventSynchronize(pl->ev[4]), "event sync");
    for (int i = 0; i < 4; ++i) CU(cudaEventElapsedTime(&out[i], pl->ev[i], pl->ev[i + 1]), "event elapsed");
    return NSFRB_OK;
}

} // extern "C"
#pragma GCC visibility pop
