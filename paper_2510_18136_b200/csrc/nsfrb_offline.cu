// Offline path of the library (nsfrb_search): the plan-specialised kernel k_search4 (nsfrb_search_kernel.cuh, compiled
// with NVRTC by nsfrb_plan_prepare or the first nsfrb_search) and the pixel-batch pipeline around it.
//
// The cube arrives as [chan][time][pixel]; the search wants one pixel's channels time-contiguous.  Instead of a second
// cube-sized buffer the plan owns two workspaces of one pixel BATCH each: k_transpose fills the first one, and every
// k_search4 launch searches batch i out of one workspace while its CTAs move batch i+1 into the other (SIDE, see the
// kernel), so the layout change of all but the first batch is hidden under the search.  Stream order between the launches
// is the only synchronisation.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "nsfrb_internal.h"

namespace nsfrb {

namespace {

const char kSearchKernelSrc[] =
#include "nsfrb_search_kernel_src.inc"
    ;

constexpr size_t kSmemLimit = 227 * 1024;
constexpr int kWmid = 80;       // widths 17..kWmid are served from the ring without a bound (it never prunes them)

// host mirror of the kernel's parameter block (nsfrb_search_kernel.cuh)
struct Search4Params {
    const float *W;
    Partial *partials;
    int32_t npix, p0, npb;
    int32_t *counter;
    float *snr_map;
    int32_t *argmax;
    float *scratch;
};

int env_int(const char *name, int dflt)
{
    const char *e = getenv(name);
    return (e && *e) ? atoi(e) : dflt;
}

void append_table(std::string &s, const char *decl, const std::vector<int> &v)
{
    s += decl;
    s += " = {";
    for (size_t i = 0; i < v.size(); ++i) {
        if (i) s += ",";
        s += std::to_string(v[i]);
    }
    s += "};\n";
}

int round_up(int v, int m) { return (v + m - 1) / m * m; }

} // namespace

struct Search4State {
    cudaLibrary_t lib = nullptr;
    cudaKernel_t fn = nullptr;
    size_t smem = 0;
    int ngroups = 0;
    int batch = 0, nbatch = 1, pxi = 1; // pixels per batch; pixels per work item
    float *W[2] = {nullptr, nullptr};
    float *scratch = nullptr;   // [grid][16][dpitch] dedispersed series of the items in flight (L2-resident)
    int grid = 0, dpitch = 0, nwarp = 16; // persistent CTAs (16 / nwarp per SM)
    int32_t *counter = nullptr; // [npix] tickets of the per-pixel reduction
    // host-cube variant (nsfrb_search_host): two device slabs [nchan][nt][batch] filled by strided copies on a copy stream
    float *slab[2] = {nullptr, nullptr};
    cudaStream_t s_copy = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_copied[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
    size_t bytes = 0;
};

namespace {

// geometry shared by the prologue and the launch: ring length, shared memory, batch size
struct Geo {
    int H, nwarp, pxi, batch, nbatch, ngroups, dpitch, sdir, prune;
    size_t smem;
};

// mirrors kSmemFloats of the kernel: rings (two planes), 8-slot and 32-slot minima twice | per-(pixel, trial) results
size_t search4_smem(int H, int nwarp, int pxi, int nt)
{
    const size_t nfl = (size_t)nwarp * ((H + 16) + 2 * (H / 8) + 2 * (H / 32)) + (size_t)pxi * nwarp * (8 + (nt + 255) / 256 + 2);
    return nfl * sizeof(float) + 64;
}

bool search4_geo(const nsfrb_plan *pl, Geo &g)
{
    // trials (= warps) per CTA: 16 by default; 24 (80 registers per thread, more latency hidden) where a power-of-two ring
    // still fits 24 warps and the last group is no emptier than with 16 -- short series with few channels (C4: 141 -> 122 ms;
    // C3 and C5 are slower with 24: 32 trials split 24 + 8, 64 channels want the registers).  NSFRB_SEARCH_WARPS overrides.
    g.nwarp = env_int("NSFRB_SEARCH_WARPS", 0);
    if (g.nwarp != 8 && g.nwarp != 16 && g.nwarp != 24 && g.nwarp != 32) {
        const int hmin0 = round_up(std::max(pl->wmax_used, 1) + kBlockLen + 32, 64);
        int hp = 64;
        while (hp < hmin0) hp <<= 1;
        const int pad16 = (pl->nuniq + 15) / 16 * 16 - pl->nuniq, pad24 = (pl->nuniq + 23) / 24 * 24 - pl->nuniq;
        const bool fits24 = search4_smem(hp, 24, 16, pl->nt) <= kSmemLimit;
        g.nwarp = (fits24 && pl->nchan <= 24 && pad24 <= pad16) ? 24 : 16;
    }
    g.ngroups = (pl->nuniq + g.nwarp - 1) / g.nwarp;
    // pixel batches: about NSFRB_SEARCH_BATCH_MB (default 1024) of workspace each, at least ~8192 items per launch
    const size_t bpp = (size_t)pl->nchan * pl->pitch * sizeof(float);
    const size_t target = (size_t)std::max(1, env_int("NSFRB_SEARCH_BATCH_MB", 1024)) << 20;
    long long nb = (long long)(target / bpp);
    nb = std::max<long long>(nb, (8192 + g.ngroups - 1) / g.ngroups);
    if (env_int("NSFRB_SEARCH_BATCH_PIX", 0) > 0) nb = env_int("NSFRB_SEARCH_BATCH_PIX", 0); // tests: force small batches
    nb = std::max<long long>(8, nb & ~7LL);
    if (nb >= pl->npix) { g.batch = pl->npix; g.nbatch = 1; }
    else { g.batch = (int)nb; g.nbatch = (pl->npix + g.batch - 1) / g.batch; }
    g.sdir = std::max(0, std::min(16, env_int("NSFRB_SEARCH_SDIR", 8)));   // widths up to here are evaluated without a bound
    g.prune = env_int("NSFRB_SEARCH_PRUNE", 1) != 0;
    g.dpitch = round_up(pl->nt, 512);
    // pixels per work item: the item's barriers are shared by them and the tail keeps one warp per pixel busy.  The scratch
    // (pxi x nwarp series per CTA) is kept to about 0.6 MB per CTA, so that the scratch of all 148 CTAs (~90 MB) stays in the
    // 126 MB L2 between sweep A, which writes it, and sweep B, which reads it three times: 2 / 12 / 1 pixels on C3 / C4 / C5
    // (measured: 2 MB per CTA, which cycles through HBM, costs +3 % / +1 % / +13 %; profiles/r02.md)
    const size_t series = (size_t)g.nwarp * g.dpitch * sizeof(float);
    g.pxi = (int)std::max<size_t>(1, std::min<size_t>(16, (640u << 10) / series));
    if (g.pxi >= 4) g.pxi &= ~3; // (whole groups of four: the tail hands a pixel to each of four warp quads)
    if (env_int("NSFRB_SEARCH_PXI", 0) > 0) g.pxi = std::min(16, env_int("NSFRB_SEARCH_PXI", 0));
    g.pxi = std::min(g.pxi, g.nwarp);
    // ring: wmax + one block + the rows the bounds read, a multiple of 64; a power of two (every wrap one AND) when shared
    // memory allows
    const size_t limit = kSmemLimit / std::max(1, 16 / g.nwarp) - (g.nwarp == 8 ? 1024 : 0);
    const int hmin = round_up(std::max(pl->wmax_used, 1) + kBlockLen + 32, 64);
    int h2 = 64;
    while (h2 < hmin) h2 <<= 1;
    g.H = search4_smem(h2, g.nwarp, g.pxi, pl->nt) <= limit ? h2 : hmin;
    if (search4_smem(g.H, g.nwarp, g.pxi, pl->nt) > limit) return false;
    g.smem = search4_smem(g.H, g.nwarp, g.pxi, pl->nt);
    return true;
}

std::string search4_prologue(const nsfrb_plan *pl, const Geo &g)
{
    std::string s = "// generated by nsfrb_offline.cu for one plan (offline kernel)\n";
    auto def = [&](const char *n, long long v) { s += "#define " + std::string(n) + " " + std::to_string(v) + "\n"; };
    def("NCHAN", pl->nchan); def("NU", pl->nuniq); def("NW", std::max(pl->nw_used, 1)); def("NWARP", g.nwarp); def("H", g.H);
    def("PITCH", pl->pitch); def("DPITCH", g.dpitch); def("NT", pl->nt); def("WMID", std::min(kWmid, g.H - kBlockLen - 32));
    def("SDIR", g.sdir); def("PXI", g.pxi); def("PRUNE", g.prune);
    s += "static __device__ constexpr short D_TAB[NU][NCHAN] = {";
    for (int u = 0; u < pl->nuniq; ++u) {
        s += u ? ",{" : "{";
        for (int ch = 0; ch < pl->nchan; ++ch) {
            if (ch) s += ",";
            s += std::to_string(pl->delays_u[(size_t)u * pl->nchan + ch]);
        }
        s += "}";
    }
    s += "};\n";
    std::vector<int> dmax(pl->dmax_u.begin(), pl->dmax_u.end()), kof(pl->k_of_u.begin(), pl->k_of_u.end());
    append_table(s, "static __device__ constexpr int DMAX_TAB[NU]", dmax);
    append_table(s, "static __device__ constexpr int K_OF_U[NU]", kof);
    std::vector<int> w(pl->widths_used.begin(), pl->widths_used.end());
    if (w.empty()) w.push_back(0x3fffffff);
    append_table(s, "static __device__ constexpr int W_TAB[NW]", w);
    std::vector<int> jw(pl->j_of_used.begin(), pl->j_of_used.end());
    if (jw.empty()) jw.push_back(0);
    append_table(s, "static __device__ constexpr int J_OF_W[NW]", jw);
    return s;
}

int fail_cuda(cudaError_t e, const char *what, std::string &err)
{
    err = std::string(what) + ": " + cudaGetErrorString(e);
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? NSFRB_ENOMEM : NSFRB_ECUDA;
}
#define OCU(call, what)                                              \
    do {                                                             \
        cudaError_t e__ = (call);                                    \
        if (e__ != cudaSuccess) return fail_cuda(e__, what, err);    \
    } while (0)

} // namespace

bool search4_usable(const nsfrb_plan *pl)
{
    const char *e = getenv("NSFRB_SEARCH_JIT");
    if (e && std::strcmp(e, "0") == 0) return false;
    Geo g;
    return pl->nw_used >= 1 && pl->nw_used <= 32 && pl->n_wb == 1 && search4_geo(pl, g);
}

int search4_source(const nsfrb_plan *pl, std::string &src, std::string &err)
{
    Geo g;
    if (pl->nw_used > 32 || !search4_geo(pl, g)) { err = "k_search4 handles at most 32 usable widths and needs its tiles to fit shared memory"; return NSFRB_EINVAL; }
    src = search4_prologue(pl, g);
    src += kSearchKernelSrc;
    return NSFRB_OK;
}

void search4_free(nsfrb_plan *p)
{
    if (!p || !p->search4) return;
    if (p->search4->lib) cudaLibraryUnload(p->search4->lib);
    cudaFree(p->search4->counter);
    cudaFree(p->search4->scratch);
    cudaFree(p->search4->W[0]);
    cudaFree(p->search4->W[1]);
    cudaFree(p->search4->slab[0]);
    cudaFree(p->search4->slab[1]);
    if (p->search4->s_copy) cudaStreamDestroy(p->search4->s_copy);
    if (p->search4->ev_fork) cudaEventDestroy(p->search4->ev_fork);
    for (int b = 0; b < 2; ++b) {
        if (p->search4->ev_copied[b]) cudaEventDestroy(p->search4->ev_copied[b]);
        if (p->search4->ev_free[b]) cudaEventDestroy(p->search4->ev_free[b]);
    }
    cudaGetLastError();
    delete p->search4;
    p->search4 = nullptr;
}

size_t search4_bytes(const nsfrb_plan *p) { return (p && p->search4) ? p->search4->bytes : 0; }
int search4_ring_len(const nsfrb_plan *pl)
{
    Geo g;
    return search4_geo(pl, g) ? g.H : pl->H;
}

// Compile the kernel and allocate the batch workspaces (nsfrb_plan_prepare; also the first nsfrb_search).
int search4_prepare(nsfrb_plan *pl, std::string &err)
{
    if (pl->search4) return NSFRB_OK;
    Geo g;
    if (!search4_geo(pl, g)) { err = "k_search4 does not fit this plan"; return NSFRB_EINVAL; }
    Search4State *s4 = new Search4State();
    pl->search4 = s4;
    std::string src, log;
    std::vector<char> cubin;
    int rc = search4_source(pl, src, err);
    if (!rc && (rc = stream_compile(src, cubin, log))) err = "k_search4 compile failed: " + log;
    if (rc) { search4_free(pl); return rc; }
    s4->ngroups = g.ngroups; s4->smem = g.smem; s4->batch = g.batch; s4->nbatch = g.nbatch; s4->pxi = g.pxi;
    cudaError_t e = cudaLibraryLoadData(&s4->lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (e == cudaSuccess) e = cudaLibraryGetKernel(&s4->fn, s4->lib, "k_search4");
    if (e == cudaSuccess) e = cudaFuncSetAttribute((const void *)s4->fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s4->smem);
    s4->nwarp = g.nwarp;
    // (+ slack: sweep A reads up to one block + the largest delay past the end of a row; the values are never used)
    const size_t wb = ((size_t)g.batch * pl->nchan * (size_t)pl->pitch + 1024 + pl->dmax_all) * sizeof(float);
    for (int b = 0; b < (g.nbatch > 1 ? 2 : 1) && e == cudaSuccess; ++b) {
        e = cudaMalloc(reinterpret_cast<void **>(&s4->W[b]), wb);
        if (e == cudaSuccess) e = cudaMemset(s4->W[b], 0, wb);
        if (e == cudaSuccess) s4->bytes += wb;
    }
    if (e == cudaSuccess) { // one CTA per SM, each with the dedispersed series of its item in flight
        int nsm = 0;
        e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, pl->device);
        s4->grid = std::max(1, nsm) * std::max(1, 16 / g.nwarp);
        s4->dpitch = g.dpitch;
        const size_t sb = (size_t)s4->grid * g.pxi * g.nwarp * g.dpitch * sizeof(float);
        if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&s4->scratch), sb);
        if (e == cudaSuccess) e = cudaMemset(s4->scratch, 0, sb);
        if (e == cudaSuccess) s4->bytes += sb;
    }
    if (e == cudaSuccess) {
        e = cudaMalloc(reinterpret_cast<void **>(&s4->counter), (size_t)pl->npix * sizeof(int32_t));
        if (e == cudaSuccess) e = cudaMemset(s4->counter, 0, (size_t)pl->npix * sizeof(int32_t));
        if (e == cudaSuccess) s4->bytes += (size_t)pl->npix * sizeof(int32_t);
    }
    if (e != cudaSuccess) {
        const int code = fail_cuda(e, "k_search4 load / workspace", err);
        search4_free(pl);
        return code;
    }
    return NSFRB_OK;
}

// a8-like layout change of the first batch + one k_search4 launch per batch; writes snr_map and argmax
int search4_launch(nsfrb_plan *pl, const float *cube, cudaStream_t st, float *snr_map, int32_t *argmax, int *launches,
                   cudaEvent_t ev_layout, std::string &err)
{
    if (int rc = search4_prepare(pl, err)) return rc;
    Search4State *s4 = pl->search4;
    const int nb = s4->batch;
    auto count = [&](int i) { return std::min(nb, pl->npix - i * nb); };
    OCU(launch_transpose(cube, s4->W[0], pl->npix, pl->nchan, pl->nt, pl->pitch, 0, count(0), st), "k_transpose launch");
    ++*launches;
    if (ev_layout) cudaEventRecord(ev_layout, st);
    for (int i = 0; i < s4->nbatch; ++i) {
        if (i + 1 < s4->nbatch) { // the next batch's layout change, stream-ordered behind the search that last read that buffer
            OCU(launch_transpose(cube, s4->W[(i + 1) & 1], pl->npix, pl->nchan, pl->nt, pl->pitch, (i + 1) * nb, count(i + 1), st),
                "k_transpose launch");
            ++*launches;
        }
        Search4Params sp;
        sp.W = s4->W[i & 1]; sp.partials = pl->d_partials; sp.npix = pl->npix; sp.p0 = i * nb; sp.npb = count(i);
        sp.counter = s4->counter; sp.snr_map = snr_map; sp.argmax = argmax; sp.scratch = s4->scratch;
        void *args[] = {&sp};
        const long long items = (long long)((sp.npb + s4->pxi - 1) / s4->pxi) * s4->ngroups;
        if (items <= 0 || items > 0x7fffffffLL) { err = "too many work items for one launch"; return NSFRB_EINVAL; }
        OCU(cudaLaunchKernel((const void *)s4->fn, dim3((unsigned)std::min<long long>(items, s4->grid)), dim3(32 * s4->nwarp), args, s4->smem, st),
            "k_search4 launch");
        ++*launches;
    }
    return NSFRB_OK;
}

// The same pipeline fed from a HOST cube (pinned memory for real overlap): batch i+1 travels host -> device slab on the copy
// stream (one strided copy: nchan*nt rows of `batch` pixels) while batch i is searched; the layout kernel reads the slab.
// No cube-sized device buffer: two slabs of one batch each.  Outputs are device buffers; the caller copies them back.
int search4_launch_host(nsfrb_plan *pl, const float *cube_host, cudaStream_t st, float *snr_map, int32_t *argmax, int *launches,
                        std::string &err)
{
    if (int rc = search4_prepare(pl, err)) return rc;
    Search4State *s4 = pl->search4;
    const int nb = s4->batch;
    auto count = [&](int i) { return std::min(nb, pl->npix - i * nb); };
    const size_t rows = (size_t)pl->nchan * pl->nt;
    if (!s4->s_copy) {
        OCU(cudaStreamCreateWithFlags(&s4->s_copy, cudaStreamNonBlocking), "copy stream");
        OCU(cudaEventCreateWithFlags(&s4->ev_fork, cudaEventDisableTiming), "event");
        for (int b = 0; b < 2; ++b) {
            OCU(cudaEventCreateWithFlags(&s4->ev_copied[b], cudaEventDisableTiming), "event");
            OCU(cudaEventCreateWithFlags(&s4->ev_free[b], cudaEventDisableTiming), "event");
        }
    }
    for (int b = 0; b < (s4->nbatch > 1 ? 2 : 1); ++b)
        if (!s4->slab[b]) {
            const size_t sb = rows * (size_t)nb * sizeof(float);
            OCU(cudaMalloc(reinterpret_cast<void **>(&s4->slab[b]), sb), "slab alloc");
            s4->bytes += sb;
        }
    OCU(cudaEventRecord(s4->ev_fork, st), "event record"); // the copies start where the caller's stream stands
    OCU(cudaStreamWaitEvent(s4->s_copy, s4->ev_fork, 0), "stream wait");
    for (int i = 0; i < s4->nbatch; ++i) {
        const int b = i & 1, n = count(i);
        if (i >= 2) OCU(cudaStreamWaitEvent(s4->s_copy, s4->ev_free[b], 0), "stream wait"); // the layout kernel of batch i-2 has read the slab
        OCU(cudaMemcpy2DAsync(s4->slab[b], (size_t)n * sizeof(float), cube_host + (size_t)i * nb, (size_t)pl->npix * sizeof(float),
                              (size_t)n * sizeof(float), rows, cudaMemcpyHostToDevice, s4->s_copy),
            "H2D batch");
        OCU(cudaEventRecord(s4->ev_copied[b], s4->s_copy), "event record");
        OCU(cudaStreamWaitEvent(st, s4->ev_copied[b], 0), "stream wait");
        // (W[b] was last read by the search of batch i-2: stream order on st)
        OCU(launch_transpose(s4->slab[b], s4->W[b], n, pl->nchan, pl->nt, pl->pitch, 0, n, st), "k_transpose launch");
        OCU(cudaEventRecord(s4->ev_free[b], st), "event record");
        ++*launches;
        Search4Params sp;
        sp.W = s4->W[b]; sp.partials = pl->d_partials; sp.npix = pl->npix; sp.p0 = i * nb; sp.npb = n;
        sp.counter = s4->counter; sp.snr_map = snr_map; sp.argmax = argmax; sp.scratch = s4->scratch;
        void *args[] = {&sp};
        const long long items = (long long)((sp.npb + s4->pxi - 1) / s4->pxi) * s4->ngroups;
        OCU(cudaLaunchKernel((const void *)s4->fn, dim3((unsigned)std::min<long long>(items, s4->grid)), dim3(32 * s4->nwarp), args, s4->smem, st),
            "k_search4 launch");
        ++*launches;
    }
    return NSFRB_OK;
}

} // namespace nsfrb
