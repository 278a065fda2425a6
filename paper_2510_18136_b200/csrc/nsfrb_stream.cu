// Real-time path of the library (nsfrb_stream_push): ring update (a8), the plan-specialised backward
// march k_stream (a1..a6, nsfrb_stream_kernel.cuh, compiled with NVRTC when the first chunk arrives) and the
// reduction of its per-slice results.  Host logic here; the device code of the march is in the .cuh.
#include <nvrtc.h>
#include <sys/stat.h>
#include <unistd.h>

#include <cerrno>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "nsfrb_internal.h"

namespace nsfrb {

namespace {

// The kernel source, embedded at build time (build.py writes the .inc from nsfrb_stream_kernel.cuh).
const char kStreamKernelSrc[] =
#include "nsfrb_stream_kernel_src.inc"
    ;

struct SPartial {
    float snr;
    int32_t k, j, t;
};

// host mirror of the kernel's parameter block (nsfrb_stream_kernel.cuh)
struct StreamParams {
    const float *ring;
    float *mu0;
    SPartial *partials;
    int32_t top_row, len, i0, C, nslice, slice0;
    float *mws;
    int32_t *aws;
    float *sws;
    int32_t bound[9];
    float *snr_cube;
    int32_t *toa_cube;
    float *sig_out;
    int32_t t_offset;
    const float *dlt;  // INCR: exact mean minus its float rounding, and 1/sigma, per (unique trial, pixel)
    const float *rsig;
    const float *dh;   // DHIST: dedispersed history [pixel block][rows][nuniq][32]
    const float *dh8;  // COARSE: its 8-row block sums [pixel block][2 * L / 8][nuniq][32]
};

// host mirror of k_stream_stats's parameter block (nsfrb_stream_kernel.cuh)
struct StatsParams {
    const float *ring;
    double *s1, *s2;
    float *mu, *dlt, *rsig, *sig_out;
    int32_t row_lo, add, first, pad;
    long long ring_lo, lo_prev, n_prev, lo, n;
    float *dh;
    float *dh8;
};

struct StreamCfg {
    int KK = 8, GPC = 2, SEG = 2, TT = 4, MINB = 1; // tile shape
    int PFD = 6;                                    // L2 prefetch distance in tiles
    int CMAX = 25;                                  // ends per pass (shared-memory budget)
    int NW = 0, NSUPER = 1;
    float light_cost = 1.0f;                        // time of a light tile relative to a plain dedispersion tile (segment balance): it waits on memory; 1.0 measured best on C2 with SEG=2 (profiles/r01_v5.md)
    int LIGHT = 1;                                  // INCR only: plain runs are summed once for all trials of a thread (light tiles)
    int INCR = 1;                                   // 1: mean/sigma kept incrementally by k_stream_stats (the march stops at the last start range)
    int COARSE = 1;                                 // DHIST only, ring length a multiple of 8: 8-row block sums of the history serve the plain runs
    int DHIST = 1;                                  // INCR only: k_stream_stats also keeps every trial's dedispersed samples (a second ring); the march reads those
    size_t smem = 0;
    int threads() const { return 32 * GPC * SEG; }
};

constexpr size_t kSmemLimit = 227 * 1024;

size_t cfg_smem(const StreamCfg &c)
{
    const size_t trials = (size_t)c.GPC * c.KK;
    const size_t qe = trials * c.CMAX * 32, sg = trials * c.SEG * 32, red = (size_t)c.GPC * 32 * 4;
    (void)sg;
    const size_t qpad = c.DHIST ? (size_t)c.TT * 32 : 0; // padding rows before and after Qe (nsfrb_stream_kernel.cuh: QPAD)
    return (qe + 2 * qpad + red + (size_t)c.GPC * c.SEG * 2) * 4;
}

// Tile shape for a plan: KK trials per thread, GPC groups x SEG segments of warps per CTA.
// dhist: 1/0 = with/without the dedispersed history, -1 = the default (NSFRB_STREAM_DHIST, else on)
bool choose_cfg(const nsfrb_plan *pl, int chunk_nt, const char *variant, StreamCfg &c, std::string &err, int dhist = -1)
{
    c = StreamCfg();
    c.NW = std::max(pl->nw_used, 1);
    int kk = 8, gpc = 2, seg = 2, tt = 2, minb = 3, pfd = 6;
    {
        const char *e = getenv("NSFRB_STREAM_STATS"); // "march": the march itself accumulates mean and variance over the whole ring (round-1 v4 behaviour)
        c.INCR = (e && std::strcmp(e, "march") == 0) ? 0 : 1;
        if (const char *lt = getenv("NSFRB_STREAM_LIGHT")) c.LIGHT = atoi(lt) != 0;
        if (!c.INCR) c.LIGHT = 0;
        if (dhist < 0) {
            const char *dh = getenv("NSFRB_STREAM_DHIST");
            dhist = dh ? (atoi(dh) != 0) : 1;
        }
        c.DHIST = (c.INCR && dhist) ? 1 : 0;
        const char *co = getenv("NSFRB_STREAM_COARSE");
        c.COARSE = (c.DHIST && c.LIGHT && pl->nt % 8 == 0 && !(co && atoi(co) == 0)) ? 1 : 0;
        if (c.COARSE && !getenv("NSFRB_STREAM_LIGHT_COST")) c.light_cost = 0.15f; // a plain tile costs one block load per 8 rows
        if (const char *lc = getenv("NSFRB_STREAM_LIGHT_COST")) c.light_cost = (float)atof(lc);
    }
    if (c.DHIST) {
        // a thread holds KK*TT history values and no raw rows, the trials of a thread share nothing and every DM group runs the
        // same instance of the code: fewer trials per thread and more warps per CTA (the shared-memory Qe block of a CTA is per
        // trial either way) -- 4 trials x 4 groups, six steps per tile (128 registers) measured best on C2 (profiles/r02.md)
        kk = 4; gpc = 4; seg = 1; tt = 6; minb = 4; pfd = 2;
    } else if (pl->nchan > 24) { // the thread holds nchan*TT raw rows in registers: one time step per tile, more registers
        tt = 1;
        minb = 2;
    } else if (c.LIGHT) {
        // light tiles wait on memory, not on the issue slots, and a second time segment only adds its imbalance: one
        // segment per CTA (64-thread CTAs, up to 255 registers) with three steps per tile and an L2 prefetch distance of
        // four tiles measured best on C2 (profiles/r01_v5.md)
        seg = 1;
        tt = 3;
        minb = 4;
        pfd = 4;
    }
    if (variant && *variant) {
        if (sscanf(variant, "%d,%d,%d,%d,%d,%d", &kk, &gpc, &seg, &tt, &minb, &pfd) < 4) {
            err = "bad k_stream variant string (want KK,GPC,SEG,TT[,MINB])";
            return false;
        }
    }
    kk = std::max(1, std::min(kk, pl->nuniq));
    const int ngroups = (pl->nuniq + kk - 1) / kk;
    gpc = std::max(1, std::min(gpc, ngroups));
    seg = std::max(1, std::min(seg, 8));
    tt = std::max(1, std::min(tt, 8));
    if (!(variant && *variant)) {
        // register estimate of the default shape: raw rows (nchan*TT) + carried halo (sum over channels of the delay
        // spread within a group of kk trials) + accumulators and state; above the 3-CTAs-per-SM budget use 2 CTAs
        int carry = 0;
        for (int g0 = 0; g0 < pl->nuniq; g0 += kk) {
            int s = 0;
            const int g1 = std::min(g0 + kk, pl->nuniq) - 1;
            for (int ch = 0; ch < pl->nchan; ++ch) {
                int lo = 1 << 30, hi = -(1 << 30);
                for (int u = g0; u <= g1; ++u) {
                    const int e = pl->dmax_u[g1] - pl->delays_u[(size_t)u * pl->nchan + ch];
                    lo = std::min(lo, e);
                    hi = std::max(hi, e);
                }
                s += hi - lo;
            }
            carry = std::max(carry, s);
        }
        // fewer CTAs per SM while the estimate exceeds the registers a thread may have at that residency
        const int est = c.DHIST ? 2 * kk * tt + 6 * kk + 40 : pl->nchan * tt + carry + kk * (tt + 4) + 36;
        const int threads = 32 * std::min(gpc, ngroups) * seg;
        while (minb > 1 && est > std::min(255, 65536 / (minb * threads)) - 5) --minb;
    }
    c.KK = kk; c.GPC = gpc; c.SEG = seg; c.TT = tt; c.PFD = std::max(0, std::min(pfd, 24 / tt)); // the ring's guard rows cover 24 rows of look-ahead
    c.NSUPER = (ngroups + gpc - 1) / gpc;
    // ends per pass: the whole first chunk if it fits one CTA's shared memory, else as many as fit (more passes)
    c.CMAX = std::max(1, std::min(chunk_nt, 255));
    while (c.CMAX > 1 && cfg_smem(c) > kSmemLimit - 2048) --c.CMAX;
    if (cfg_smem(c) > kSmemLimit - 2048) {
        err = "k_stream does not fit shared memory (too many widths for the tile shape)";
        return false;
    }
    c.smem = cfg_smem(c);
    const int per_sm = (int)std::min<size_t>(kSmemLimit / (c.smem + 1024), 2048 / c.threads());
    c.MINB = minb > 0 ? minb : std::max(1, std::min(per_sm, 16)); // CTAs per SM the shared memory allows
    return true;
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

std::string make_prologue(const nsfrb_plan *pl, const StreamCfg &c)
{
    std::string s = "// generated by nsfrb_stream.cu for one plan\n";
    auto def = [&](const char *n, long long v) { s += "#define " + std::string(n) + " " + std::to_string(v) + "\n"; };
    def("NPIX", pl->npix); def("NCHAN", pl->nchan); def("NU", pl->nuniq); def("KK", c.KK); def("GPC", c.GPC);
    def("SEG", c.SEG); def("TT", c.TT); def("NW", c.NW); def("CMAX", c.CMAX); def("NSUPER", c.NSUPER); def("MINB", c.MINB); def("PFD", c.PFD); def("INCR", c.INCR); def("LIGHT", c.LIGHT); def("NW_ALL", pl->nw); def("ROWS", 2 * (pl->dmax_all + 40) + 2 * pl->nt);
    def("COARSE", c.COARSE); def("DHIST", c.DHIST); def("LRING", pl->nt); def("GUARD", pl->dmax_all + 40);
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
    std::vector<int> w, j;
    for (int i : pl->stream_worder) {
        w.push_back(pl->widths_used[i]);
        j.push_back(pl->j_of_used[i]);
    }
    if (w.empty()) { w.push_back(0x3fffffff); j.push_back(0); } // no usable width: one that never has a cell
    append_table(s, "static __device__ constexpr int W_TAB[NW]", w);
    append_table(s, "static __device__ constexpr int J_OF_W[NW]", j);
    s += "static __device__ constexpr float RSQ_W[NW] = {";
    for (size_t i = 0; i < w.size(); ++i) {
        char buf[64];
        snprintf(buf, sizeof buf, "%s%.9ef", i ? "," : "", 1.0 / std::sqrt((double)w[i]));
        s += buf;
    }
    s += "};\n";
    return s;
}

} // namespace

int stream_source(const nsfrb_plan *pl, int chunk_nt, const char *variant, std::string &src, std::string &err)
{
    StreamCfg c;
    if (!choose_cfg(pl, chunk_nt, variant, c, err)) return NSFRB_ENOMEM;
    src = make_prologue(pl, c);
    src += "#define CUBES 0\n";
    src += kStreamKernelSrc;
    return NSFRB_OK;
}

namespace {

// Optional on-disk cache of compiled kernels, keyed by a hash of the generated source and the NVRTC version
// (NSFRB_JIT_CACHE=<dir> to place it, NSFRB_JIT_CACHE=0 to switch it off; default /tmp/nsfrb_jit_cache_<uid>, mode 0700).
std::string cache_path(const std::string &src)
{
    const char *dir = getenv("NSFRB_JIT_CACHE");
    if (dir && std::strcmp(dir, "0") == 0) return "";
    // default: a private per-user directory (a cubin read from the cache is executed: nobody else may write there)
    std::string d = (dir && *dir) ? dir : "/tmp/nsfrb_jit_cache_" + std::to_string((long long)geteuid());
    if (mkdir(d.c_str(), 0700) != 0 && errno != EEXIST) return ""; // one level; no cache if it cannot be made
    struct stat sb;
    if (lstat(d.c_str(), &sb) != 0 || !S_ISDIR(sb.st_mode) || sb.st_uid != geteuid() || (sb.st_mode & (S_IWGRP | S_IWOTH)))
        return ""; // not a directory of ours (or writable by others): compile every time instead
    int major = 0, minor = 0;
    nvrtcVersion(&major, &minor);
    uint64_t h = 1469598103934665603ull; // FNV-1a
    for (unsigned char ch : src) { h ^= ch; h *= 1099511628211ull; }
    h ^= (uint64_t)(major * 100 + minor); h *= 1099511628211ull;
    char name[64];
    snprintf(name, sizeof name, "/k_%016llx_%zu.cubin", (unsigned long long)h, src.size());
    return d + name;
}

} // namespace

int stream_compile(const std::string &src, std::vector<char> &cubin, std::string &log)
{
    const std::string cpath = cache_path(src);
    if (!cpath.empty()) {
        if (FILE *f = fopen(cpath.c_str(), "rb")) {
            fseek(f, 0, SEEK_END);
            const long n = ftell(f);
            fseek(f, 0, SEEK_SET);
            cubin.resize(n > 0 ? (size_t)n : 0);
            const size_t got = n > 0 ? fread(cubin.data(), 1, (size_t)n, f) : 0;
            fclose(f);
            if (n > 4 && got == (size_t)n && std::memcmp(cubin.data(), "\x7f" "ELF", 4) == 0) {
                log = "cached: " + cpath;
                return NSFRB_OK;
            }
        }
    }
    nvrtcProgram prog;
    if (nvrtcCreateProgram(&prog, src.c_str(), "nsfrb_k_stream.cu", 0, nullptr, nullptr) != NVRTC_SUCCESS) {
        log = "nvrtcCreateProgram failed";
        return NSFRB_ECUDA;
    }
    const char *opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", "-default-device"};
    const nvrtcResult r = nvrtcCompileProgram(prog, 4, opts);
    size_t ls = 0;
    nvrtcGetProgramLogSize(prog, &ls);
    log.assign(ls, '\0');
    if (ls) nvrtcGetProgramLog(prog, &log[0]);
    if (r != NVRTC_SUCCESS) {
        nvrtcDestroyProgram(&prog);
        log = std::string("NVRTC: ") + nvrtcGetErrorString(r) + "\n" + log;
        return NSFRB_ECUDA;
    }
    size_t cs = 0;
    nvrtcGetCUBINSize(prog, &cs);
    cubin.resize(cs);
    nvrtcGetCUBIN(prog, cubin.data());
    nvrtcDestroyProgram(&prog);
    if (cs && !cpath.empty()) { // write-then-rename so that a concurrent reader never sees a partial file
        const std::string tmp = cpath + ".tmp" + std::to_string((long long)getpid());
        if (FILE *f = fopen(tmp.c_str(), "wb")) {
            const bool ok = fwrite(cubin.data(), 1, cs, f) == cs;
            fclose(f);
            if (!ok || rename(tmp.c_str(), cpath.c_str()) != 0) remove(tmp.c_str());
        }
    }
    return cs ? NSFRB_OK : NSFRB_ECUDA;
}

// ------------------------------------------------------------------------------------------------
// device state of the real-time path and the small kernels around k_stream
// ------------------------------------------------------------------------------------------------
struct StreamState {
    StreamCfg cfg;
    cudaLibrary_t lib[2] = {nullptr, nullptr}; // [0] plain, [1] with the cube outputs compiled in
    cudaKernel_t fn[2] = {nullptr, nullptr};
    cudaKernel_t fn_stats[2] = {nullptr, nullptr}; // k_stream_stats of the same module (INCR)
    float *ring = nullptr; // [pixel block][G + 2L + G][nchan][32]
    float *dhist = nullptr; // [pixel block][G + 2L + G][nuniq][32]  dedispersed history (cfg.DHIST)
    float *dh8 = nullptr;   // [pixel block][2L/8][nuniq][32]  its 8-row block sums (cfg.COARSE)
    float *base = nullptr; // [nchan][npix]  first sample ever, removed from every stored sample
    float *mu0 = nullptr;  // [nuniq][npix]
    // incremental statistics (k_stream_stats): float64 sums of D and D^2 over the valid samples of every (unique trial,
    // pixel), and what k_stream's reduction needs of them
    double *st1 = nullptr, *st2 = nullptr;
    float *dlt = nullptr, *rsig = nullptr;
    SPartial *partials = nullptr;
    float *mws = nullptr;  // running maxima per (pixel block, supergroup, trial, width, lane)
    int32_t *aws = nullptr;
    float *sws = nullptr;  // segment totals
    float *snr_cube = nullptr; // caller's optional [ndm][nwidth][npix] outputs (nsfrb_stream_set_cubes)
    int32_t *toa_cube = nullptr;
    int32_t *d_canon = nullptr; // [ndm] lowest dm index with the same delay vector
    // running-sigma mode (nsfrb_stream_set_running_sigma): this push's sigma and the running variance of every
    // (unique trial, pixel); cubes owned by the library when the caller registered none
    float *sig = nullptr, *var = nullptr;
    bool var_init = false;
    float *own_cs = nullptr;
    int32_t *own_ct = nullptr;
    int guard = 0, max_slices = 0;
    size_t bytes = 0;
};

namespace {

// base[c][p] = the lower median of the first min(chunk_nt, 32) samples of the first chunk (reading R32): the stored level every
// ring value is taken relative to.  It cancels in D - mu; it only has to be NEAR the data so that float32 storage keeps
// its resolution -- a single outlier (the very first sample, say) must not become the reference.
__global__ void __launch_bounds__(256) k_stream_base(const float *__restrict__ chunk, float *__restrict__ base, int npix, int chunk_nt)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (p >= npix) return;
    const int m = chunk_nt < 32 ? chunk_nt : 32;
    const float *src = chunk + (size_t)c * chunk_nt * npix + p;
    float v[32];
    for (int i = 0; i < m; ++i) v[i] = src[(size_t)i * npix];
    float med = v[0];
    for (int i = 0; i < m; ++i) { // the element with exactly (m - 1) / 2 elements before it in (value, index) order
        int rank = 0;
        for (int j = 0; j < m; ++j) rank += (v[j] < v[i]) || (v[j] == v[i] && j < i);
        if (rank == (m - 1) / 2) med = v[i];
    }
    if (!(med == med) || fabsf(med) > 3.0e38f) med = 0.f; // non-finite data: no reference level
    base[(size_t)c * npix + p] = med;
}

// a8: chunk[c][i][p] - base[c][p] -> ring[p/32][guard + slot (and + L)][c][p%32], slot = (slot0 + i) mod L
template <typename V>
__global__ void __launch_bounds__(256) k_stream_push(const V *__restrict__ chunk, V *__restrict__ ring, V *__restrict__ base,
                                                      int npv, int nchan, int chunk_nt, int L, int guard, int rows, int slot0,
                                                      int set_base)
{
    constexpr int kPer = 32 / (int)(sizeof(V) / 4); // vectors per 32-pixel block
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (p >= npv) return;
    const V *src = chunk + (size_t)c * chunk_nt * npv + p;
    V b;
    if (set_base) {
        b = src[0];
        base[(size_t)c * npv + p] = b;
    } else {
        b = base[(size_t)c * npv + p];
    }
    const int pb = p / kPer, pl = p - pb * kPer;
    for (int i = blockIdx.z; i < chunk_nt; i += gridDim.z) {
        V v = src[(size_t)i * npv];
        if constexpr (sizeof(V) == 16) { v.x -= b.x; v.y -= b.y; v.z -= b.z; v.w -= b.w; }
        else v -= b;
        int slot = slot0 + i;
        if (slot >= L) slot -= L;
        V *dst = ring + (((size_t)pb * rows + guard + slot) * nchan + c) * kPer + pl;
        dst[0] = v;
        dst[(size_t)L * nchan * kPer] = v;
    }
}



__device__ __forceinline__ bool sbetter(const SPartial &a, const SPartial &b)
{
    if (a.k < 0) return false;
    if (b.k < 0) return true;
    if (a.snr != b.snr) return a.snr > b.snr;
    if (a.k != b.k) return a.k < b.k;
    if (a.j != b.j) return a.j < b.j;
    return a.t < b.t;
}

// a6, last step: best slice of every pixel -> snr_map, argmax (t made absolute)
__global__ void __launch_bounds__(256) k_stream_finalize(const SPartial *__restrict__ partials, int nslice, int npix,
                                                          int t_offset, float *__restrict__ snr_map, int32_t *__restrict__ argmax)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npix) return;
    SPartial b = partials[(size_t)p * nslice];
    for (int s = 1; s < nslice; ++s) {
        const SPartial c = partials[(size_t)p * nslice + s];
        if (sbetter(c, b)) b = c;
    }
    if (b.k < 0) {
        snr_map[p] = __int_as_float(0xff800000);
        argmax[p] = -1; argmax[(size_t)npix + p] = -1; argmax[2 * (size_t)npix + p] = -1;
    } else {
        snr_map[p] = b.snr;
        argmax[p] = b.k;
        argmax[(size_t)npix + p] = b.j;
        argmax[2 * (size_t)npix + p] = (int32_t)(((uint32_t)t_offset + (uint32_t)b.t) & 0x7fffffffu);
    }
}

// Running standard deviation (reading R30): v_n = (1 - alpha) v_{n-1} + alpha sigma_n^2 per (unique trial, pixel),
// S_run = S * sigma_n / sqrt(v_n) applied to the per-(trial, width) maxima of this push (a positive factor per trial, so
// the maximising window of every (trial, width) is unchanged); then the O6 reduction over trials and widths.
__global__ void __launch_bounds__(256) k_running(const float *__restrict__ snr_cube, const int32_t *__restrict__ toa_cube,
                                                  const float *__restrict__ sig, float *__restrict__ var,
                                                  const int32_t *__restrict__ k_of_u, int nuniq, int nw, int npix,
                                                  float alpha, int first, float *__restrict__ snr_run,
                                                  int32_t *__restrict__ arg_run)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npix) return;
    float bs = __int_as_float(0xff800000);
    int bk = -1, bj = -1, bt = -1;
    for (int u = 0; u < nuniq; ++u) {
        const float s = sig[(size_t)u * npix + p];
        float v = var[(size_t)u * npix + p];
        if (s != s) continue;                      // no valid sample of this trial yet: state untouched, no window
        const float s2 = s * s;
        v = (first || v != v) ? s2 : (1.f - alpha) * v + alpha * s2;
        var[(size_t)u * npix + p] = v;
        const float sr = sqrtf(v);
        const float a = sr > 0.f ? s / sr : 0.f;   // sigma_run = 0 => S = 0 (the O5 convention)
        const int k = k_of_u[u];
        for (int j = 0; j < nw; ++j) {
            const size_t ci = ((size_t)k * nw + j) * npix + p;
            const float S = snr_cube[ci];
            if (S == __int_as_float(0xff800000)) continue;
            const float Sr = S * a;
            const int t = toa_cube[ci];
            bool better = bk < 0;
            if (!better) {
                if (Sr != bs) better = Sr > bs;
                else if (k != bk) better = k < bk;
                else if (j != bj) better = j < bj;
                else better = t < bt;
            }
            if (better) { bs = Sr; bk = k; bj = j; bt = t; }
        }
    }
    snr_run[p] = bs;
    arg_run[p] = bk;
    arg_run[(size_t)npix + p] = bj;
    arg_run[2 * (size_t)npix + p] = bt;
}

// cubes: every entry starts as "no window" (-inf, -1) ...
__global__ void __launch_bounds__(256) k_cube_fill(float *__restrict__ snr_cube, int32_t *__restrict__ toa_cube, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { snr_cube[i] = __int_as_float(0xff800000); toa_cube[i] = -1; }
}
// ... and trials with the delay vector of an earlier one repeat its planes (k_stream searches unique trials only)
__global__ void __launch_bounds__(256) k_cube_dups(float *__restrict__ snr_cube, int32_t *__restrict__ toa_cube,
                                                   const int32_t *__restrict__ canon, size_t plane)
{
    const int k = blockIdx.y, ck = canon[k];
    if (ck == k) return;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < plane) {
        snr_cube[(size_t)k * plane + i] = snr_cube[(size_t)ck * plane + i];
        toa_cube[(size_t)k * plane + i] = toa_cube[(size_t)ck * plane + i];
    }
}

inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

// Segment boundaries of one pass: multiples of TT, >= the end zone, never inside a width's start range.
void segment_bounds(const nsfrb_plan *pl, const StreamCfg &c, int len, int i0, int C, int32_t bound[9])
{
    int Rtot = std::max(0, len - pl->dmin_all);
    // INCR: mean and sigma come from k_stream_stats, so nothing lies beyond the last start range (own step
    // w + i0 + C - 1 of the widest width; a trial's group step is never ahead of its own step)
    if (c.INCR) Rtot = std::min(Rtot, std::max(pl->wmax_used, 0) + i0 + C);
    const int Rceil = round_up(Rtot, c.TT);
    for (int q = 0; q <= 8; ++q) bound[q] = Rceil;
    bound[0] = 0;
    const int lo = std::min(Rceil, round_up(i0 + C, c.TT));
    const int spread = pl->dmax_all - pl->dmin_all; // bound on delta_u = DMAXG - dmax_u
    auto cuts = [&](int b) {
        for (int i = 0; i < pl->nw_used; ++i) {
            // start range of the width in any trial's group frame: [w+i0-spread, w+i0+C-1]
            const int a = pl->widths_used[i] + i0, z = a + C - 1;
            if (a - spread <= b && b < z) return true;
        }
        return false;
    };
    // cost of every tile: 1 for the dedispersion + ~0.7 per width whose start range meets it; the boundaries
    // sit at equal shares of the total cost so that the segments of a CTA finish together
    const int ntile = Rceil / c.TT;
    std::vector<float> cum(ntile + 1, 0.f);
    for (int t = 0; t < ntile; ++t) {
        const int r0 = t * c.TT + 1, r1 = (t + 1) * c.TT + spread; // own-frame steps the tile can touch
        float cost = 1.f + (r0 <= i0 + C ? 0.5f : 0.f);
        bool met = r0 <= i0 + C;
        for (int i = 0; i < pl->nw_used; ++i) {
            const int a = pl->widths_used[i] + i0, z = a + C - 1;
            if (a <= r1 && z >= r0) { cost += 0.7f; met = true; }
        }
        if (c.LIGHT && !met) cost = c.light_cost; // a light tile (plain run): the trials share one sum of the rows
        cum[t + 1] = cum[t] + cost;
    }
    for (int q = 1; q < c.SEG; ++q) {
        const int floor_b = std::max(bound[q - 1], lo);
        const float want = cum[ntile] * q / c.SEG;
        int t = (int)(std::lower_bound(cum.begin(), cum.end(), want) - cum.begin());
        const int ideal = std::max(floor_b, std::min(Rceil, t * c.TT));
        int best = Rceil;
        for (int d = 0; d <= Rceil; d += c.TT) {
            const int up = ideal + d, dn = ideal - d;
            if (dn >= floor_b && dn <= Rceil && !cuts(dn)) { best = dn; break; }
            if (up <= Rceil && !cuts(up)) { best = up; break; }
            if (dn < floor_b && up > Rceil) break;
        }
        bound[q] = best;
    }
}

int fail_cuda(cudaError_t e, const char *what, std::string &err)
{
    err = std::string(what) + ": " + cudaGetErrorString(e);
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? NSFRB_ENOMEM : NSFRB_ECUDA;
}
#define SCU(call, what)                                              \
    do {                                                             \
        cudaError_t e__ = (call);                                    \
        if (e__ != cudaSuccess) return fail_cuda(e__, what, err);    \
    } while (0)

// Compile and load the kernel variant `cubes` (0/1) of the plan if it is not there yet.
int stream_kernel(nsfrb_plan *pl, StreamState *ss, int cubes, std::string &err)
{
    if (ss->fn[cubes]) return NSFRB_OK;
    std::string src = make_prologue(pl, ss->cfg);
    src += "#define CUBES " + std::to_string(cubes) + "\n";
    src += kStreamKernelSrc;
    std::vector<char> cubin;
    std::string log;
    if (int rc = stream_compile(src, cubin, log)) {
        err = "k_stream compile failed: " + log;
        return rc;
    }
    SCU(cudaLibraryLoadData(&ss->lib[cubes], cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0), "cudaLibraryLoadData(k_stream)");
    SCU(cudaLibraryGetKernel(&ss->fn[cubes], ss->lib[cubes], "k_stream"), "cudaLibraryGetKernel(k_stream)");
    SCU(cudaFuncSetAttribute((const void *)ss->fn[cubes], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ss->cfg.smem),
        "k_stream shared-memory attribute");
    if (ss->cfg.INCR) SCU(cudaLibraryGetKernel(&ss->fn_stats[cubes], ss->lib[cubes], "k_stream_stats"), "cudaLibraryGetKernel(k_stream_stats)");
    return NSFRB_OK;
}

int stream_init(nsfrb_plan *pl, int chunk_nt, std::string &err)
{
    StreamState *ss = new StreamState();
    pl->stream = ss;
    if (!choose_cfg(pl, chunk_nt, getenv("NSFRB_STREAM_VARIANT"), ss->cfg, err)) return NSFRB_ENOMEM;
    ss->guard = pl->dmax_all + 40;
    const size_t row = (size_t)pl->nchan * pl->npix;
    const size_t ring_b = (size_t)((pl->npix + 31) / 32) * (2 * ss->guard + 2 * pl->nt) * pl->nchan * 32 * sizeof(float);
    SCU(cudaMalloc(reinterpret_cast<void **>(&ss->ring), ring_b), "ring alloc");
    SCU(cudaMemset(ss->ring, 0, ring_b), "ring clear");
    size_t dh_b = 0;
    if (ss->cfg.DHIST) {
        dh_b = ring_b / pl->nchan * pl->nuniq;
        size_t fr = 0, tot = 0;
        // the history is a second ring, nuniq / nchan times the first: where it does not fit comfortably the march dedisperses
        if (cudaMemGetInfo(&fr, &tot) != cudaSuccess || dh_b > fr / 2) {
            cudaGetLastError();
            dh_b = 0;
            if (!choose_cfg(pl, chunk_nt, getenv("NSFRB_STREAM_VARIANT"), ss->cfg, err, 0)) return NSFRB_ENOMEM;
        } else {
            SCU(cudaMalloc(reinterpret_cast<void **>(&ss->dhist), dh_b), "dedispersed-history alloc");
            SCU(cudaMemset(ss->dhist, 0, dh_b), "dedispersed-history clear");
            if (ss->cfg.COARSE) {
                const size_t d8 = (size_t)((pl->npix + 31) / 32) * (2 * pl->nt / 8) * pl->nuniq * 32 * sizeof(float);
                SCU(cudaMalloc(reinterpret_cast<void **>(&ss->dh8), d8), "history block-sum alloc");
                SCU(cudaMemset(ss->dh8, 0, d8), "history block-sum clear");
                dh_b += d8;
            }
        }
    }
    SCU(cudaMalloc(reinterpret_cast<void **>(&ss->base), row * sizeof(float)), "base alloc");
    const size_t mu_b = (size_t)pl->nuniq * pl->npix * sizeof(float);
    SCU(cudaMalloc(reinterpret_cast<void **>(&ss->mu0), mu_b), "mu0 alloc");
    SCU(cudaMemset(ss->mu0, 0, mu_b), "mu0 clear");
    size_t st_b = 0;
    if (ss->cfg.INCR) {
        st_b = 2 * mu_b * 2 + 2 * mu_b;
        SCU(cudaMalloc(reinterpret_cast<void **>(&ss->st1), 2 * mu_b), "statistics alloc");
        SCU(cudaMalloc(reinterpret_cast<void **>(&ss->st2), 2 * mu_b), "statistics alloc");
        SCU(cudaMalloc(reinterpret_cast<void **>(&ss->dlt), mu_b), "statistics alloc");
        SCU(cudaMalloc(reinterpret_cast<void **>(&ss->rsig), mu_b), "statistics alloc");
    }
    const size_t m_b = (size_t)((pl->npix + 31) / 32) * ss->cfg.NSUPER * ss->cfg.GPC * ss->cfg.KK * ss->cfg.NW * 32 * sizeof(float);
    SCU(cudaMalloc(reinterpret_cast<void **>(&ss->mws), m_b), "maxima workspace alloc");
    SCU(cudaMalloc(reinterpret_cast<void **>(&ss->aws), m_b), "arg workspace alloc");
    const size_t s_b = (size_t)((pl->npix + 31) / 32) * ss->cfg.NSUPER * 2 * ss->cfg.GPC * ss->cfg.KK * ss->cfg.SEG * 32 * sizeof(float);
    SCU(cudaMalloc(reinterpret_cast<void **>(&ss->sws), s_b), "segment-total workspace alloc");
    {
        std::vector<int32_t> canon(pl->ndm);
        for (int k = 0; k < pl->ndm; ++k) {
            canon[k] = k;
            for (int k2 = 0; k2 < k; ++k2)
                if (std::memcmp(&pl->delays[(size_t)k2 * pl->nchan], &pl->delays[(size_t)k * pl->nchan], sizeof(int32_t) * pl->nchan) == 0) {
                    canon[k] = k2;
                    break;
                }
        }
        SCU(cudaMalloc(reinterpret_cast<void **>(&ss->d_canon), canon.size() * sizeof(int32_t)), "canon alloc");
        SCU(cudaMemcpy(ss->d_canon, canon.data(), canon.size() * sizeof(int32_t), cudaMemcpyHostToDevice), "canon upload");
    }
    ss->snr_cube = pl->cube_snr;
    ss->toa_cube = pl->cube_toa;
    ss->bytes = ring_b + dh_b + row * sizeof(float) + mu_b + 2 * m_b + s_b + st_b;
    return NSFRB_OK;
}

} // namespace

void stream_free(nsfrb_plan *p)
{
    if (!p || !p->stream) return;
    StreamState *ss = p->stream;
    cudaFree(ss->ring); cudaFree(ss->dhist); cudaFree(ss->dh8); cudaFree(ss->base); cudaFree(ss->mu0); cudaFree(ss->partials); cudaFree(ss->mws); cudaFree(ss->aws); cudaFree(ss->sws); cudaFree(ss->d_canon);
    cudaFree(ss->st1); cudaFree(ss->st2); cudaFree(ss->dlt); cudaFree(ss->rsig);
    cudaFree(ss->sig); cudaFree(ss->var); cudaFree(ss->own_cs); cudaFree(ss->own_ct);
    for (auto &l : ss->lib) if (l) cudaLibraryUnload(l);
    cudaGetLastError();
    delete ss;
    p->stream = nullptr;
}

// Register (or clear, with nulls) the caller's cube outputs; they are written by every later push.
int stream_set_cubes(nsfrb_plan *pl, float *snr_cube, int32_t *toa_cube, std::string &err)
{
    if ((snr_cube == nullptr) != (toa_cube == nullptr)) { err = "snr_cube and toa_cube must both be given or both be null"; return NSFRB_EINVAL; }
    pl->cube_snr = snr_cube;
    pl->cube_toa = toa_cube;
    if (pl->stream) { pl->stream->snr_cube = snr_cube; pl->stream->toa_cube = toa_cube; }
    return NSFRB_OK;
}

size_t stream_bytes(const nsfrb_plan *p) { return (p && p->stream) ? p->stream->bytes : 0; }

int stream_mode(const nsfrb_plan *p)
{
    if (!p || !p->stream) return 0;
    const StreamCfg &c = p->stream->cfg;
    return c.DHIST ? (c.COARSE ? 3 : 2) : 1;
}

void stream_reset(nsfrb_plan *p)
{
    if (!p || !p->stream) return;
    if (p->stream->mu0) cudaMemset(p->stream->mu0, 0, (size_t)p->nuniq * p->npix * sizeof(float));
    p->stream->var_init = false;   // the running variance starts again with the next push
}

// Running-sigma outputs (nulls switch the mode off).  The running variance restarts.
int stream_set_running(nsfrb_plan *pl, double alpha, float *snr_run, int32_t *arg_run, std::string &err)
{
    if ((snr_run == nullptr) != (arg_run == nullptr)) { err = "snr_map_run and argmax_run must both be given or both be null"; return NSFRB_EINVAL; }
    if (snr_run && !(alpha > 0.0 && alpha <= 1.0)) { err = "alpha must be in (0, 1]"; return NSFRB_EINVAL; }
    pl->run_alpha = (float)alpha;
    pl->run_snr = snr_run;
    pl->run_arg = arg_run;
    if (pl->stream) pl->stream->var_init = false;
    return NSFRB_OK;
}

// Ring, statistics and workspaces + the compiled kernel for chunks of chunk_nt samples (nsfrb_plan_prepare).
int stream_prepare(nsfrb_plan *pl, int chunk_nt, std::string &err)
{
    if (!pl->stream) {
        if (int rc = stream_init(pl, chunk_nt, err)) {
            stream_free(pl);
            return rc;
        }
    }
    return stream_kernel(pl, pl->stream, (pl->cube_snr || pl->run_snr) ? 1 : 0, err);
}

int stream_push(nsfrb_plan *pl, const float *chunk, int chunk_nt, cudaStream_t st, float *snr_map, int32_t *argmax,
                int *launches, std::string &err)
{
    if (!pl->stream) {
        if (int rc = stream_init(pl, chunk_nt, err)) {
            stream_free(pl);
            return rc;
        }
    }
    StreamState *ss = pl->stream;
    if (chunk_nt > ss->cfg.CMAX) {
        // a longer chunk than the kernel was compiled for would run ceil(chunk_nt / CMAX) passes per push: compile for
        // the longer one instead (CMAX is the only shape parameter that depends on the chunk; the workspaces do not)
        StreamCfg c2;
        std::string e2;
        if (choose_cfg(pl, chunk_nt, getenv("NSFRB_STREAM_VARIANT"), c2, e2, ss->cfg.DHIST) && c2.CMAX > ss->cfg.CMAX) {
            SCU(cudaStreamSynchronize(st), "stream sync before the kernel is replaced");
            for (int v = 0; v < 2; ++v) {
                if (ss->lib[v]) cudaLibraryUnload(ss->lib[v]);
                ss->lib[v] = nullptr; ss->fn[v] = nullptr; ss->fn_stats[v] = nullptr;
            }
            ss->cfg = c2;
        }
    }
    const bool running = pl->run_snr != nullptr;
    if (running) {   // needs this push's sigma per (unique trial, pixel) and the per-(trial, width) maxima
        const size_t nb = (size_t)pl->nuniq * pl->npix * sizeof(float);
        if (!ss->sig) {
            SCU(cudaMalloc(reinterpret_cast<void **>(&ss->sig), nb), "sigma alloc");
            SCU(cudaMalloc(reinterpret_cast<void **>(&ss->var), nb), "running variance alloc");
            ss->bytes += 2 * nb;
            ss->var_init = false;
        }
        if (!ss->snr_cube && !ss->own_cs) {
            const size_t cb = (size_t)pl->ndm * pl->nw * pl->npix * sizeof(float);
            SCU(cudaMalloc(reinterpret_cast<void **>(&ss->own_cs), cb), "cube alloc");
            SCU(cudaMalloc(reinterpret_cast<void **>(&ss->own_ct), cb), "cube alloc");
            ss->bytes += 2 * cb;
        }
    }
    float *const cs = ss->snr_cube ? ss->snr_cube : (running ? ss->own_cs : nullptr);
    int32_t *const ct = ss->snr_cube ? ss->toa_cube : (running ? ss->own_ct : nullptr);
    const int variant = cs ? 1 : 0;
    if (int rc = stream_kernel(pl, ss, variant, err)) return rc;
    const StreamCfg &c = ss->cfg;
    const int L = pl->nt;
    const int64_t n_prev = pl->n_received, n = n_prev + chunk_nt;
    const int64_t lo = std::max<int64_t>(0, n - L);
    const int len = (int)(n - lo);

    // ---- a1, a3 (INCR), first half: the samples that leave the valid sets, while their raw rows are still in the ring
    const int64_t lo_prev = std::max<int64_t>(0, n_prev - L);
    StatsParams tp;
    tp.ring = ss->ring; tp.s1 = ss->st1; tp.s2 = ss->st2; tp.mu = ss->mu0; tp.dlt = ss->dlt; tp.rsig = ss->rsig; tp.sig_out = nullptr;
    tp.dh = ss->dhist; tp.dh8 = ss->dh8; tp.pad = 0; tp.lo_prev = lo_prev; tp.n_prev = n_prev; tp.lo = lo; tp.n = n;
    int stat_warps = 8; // trials (warps) per CTA of k_stream_stats
    if (const char *e = getenv("NSFRB_STREAM_STATS_WARPS")) stat_warps = std::max(1, std::min(8, atoi(e)));
    const dim3 stat_grid((pl->npix + 31) / 32, (pl->nuniq + stat_warps - 1) / stat_warps), stat_block(32 * stat_warps);
    if (c.INCR && !c.DHIST && lo > lo_prev && n_prev > 0) { // (DHIST: the leaving samples come from the history, in the launch below)
        tp.row_lo = ss->guard + (int)(lo_prev % L); tp.ring_lo = lo_prev; tp.add = 0; tp.first = 0;
        void *args[] = {&tp};
        SCU(cudaLaunchKernel((const void *)ss->fn_stats[variant], stat_grid, stat_block, args, 0, st), "k_stream_stats launch");
        ++*launches;
    }
    // ---- a8: ring update
    if (n_prev == 0) { // the reference level of every (channel, pixel), from the first chunk
        dim3 grid((pl->npix + 255) / 256, pl->nchan);
        k_stream_base<<<grid, 256, 0, st>>>(chunk, ss->base, pl->npix, chunk_nt);
        SCU(cudaGetLastError(), "k_stream_base launch");
        ++*launches;
    }
    {
        const bool v4 = (pl->npix % 4 == 0) && ((reinterpret_cast<uintptr_t>(chunk) & 15u) == 0);
        const int npv = v4 ? pl->npix / 4 : pl->npix;
        const int rows = 2 * ss->guard + 2 * L;
        dim3 grid((npv + 255) / 256, pl->nchan, std::min(chunk_nt, 32));
        if (v4)
            k_stream_push<float4><<<grid, 256, 0, st>>>(reinterpret_cast<const float4 *>(chunk), reinterpret_cast<float4 *>(ss->ring),
                                                        reinterpret_cast<float4 *>(ss->base), npv, pl->nchan, chunk_nt, L, ss->guard, rows,
                                                        (int)(n_prev % L), 0);
        else
            k_stream_push<float><<<grid, 256, 0, st>>>(chunk, ss->ring, ss->base, npv, pl->nchan, chunk_nt, L, ss->guard, rows,
                                                       (int)(n_prev % L), 0);
        SCU(cudaGetLastError(), "k_stream_push launch");
        ++*launches;
    }
    pl->n_received = n;
    if (c.INCR) { // second half: the samples that enter; mean, 1/sigma (and sigma itself for the running-sigma mode)
        tp.row_lo = ss->guard + (int)(lo % L); tp.ring_lo = lo; tp.add = c.DHIST ? 2 : 1; tp.first = n_prev == 0 ? 1 : 0;
        tp.sig_out = running ? ss->sig : nullptr;
        void *args[] = {&tp};
        SCU(cudaLaunchKernel((const void *)ss->fn_stats[variant], stat_grid, stat_block, args, 0, st), "k_stream_stats launch");
        ++*launches;
    }
    if (pl->profiling && pl->ev[1]) cudaEventRecord(pl->ev[1], st);

    // ---- k_stream: one pass per batch of CMAX ends
    const int npass = (chunk_nt + c.CMAX - 1) / c.CMAX;
    const int nslice = npass * c.NSUPER;
    if (nslice > ss->max_slices) {
        cudaFree(ss->partials);
        ss->partials = nullptr;
        ss->max_slices = 0;
        SCU(cudaMalloc(reinterpret_cast<void **>(&ss->partials), (size_t)pl->npix * nslice * sizeof(SPartial)), "partials alloc");
        ss->max_slices = nslice;
    }
    const int base_slot = (int)(lo % L);
    const size_t cube_plane = (size_t)pl->nw * pl->npix; // one trial's [nwidth][npix]
    if (cs) {
        const size_t ncube = cube_plane * pl->ndm;
        k_cube_fill<<<(unsigned)((ncube + 255) / 256), 256, 0, st>>>(cs, ct, ncube);
        SCU(cudaGetLastError(), "k_cube_fill launch");
        ++*launches;
    }
    if (running && !c.INCR)   // NaN = "this trial has no valid sample yet"
        SCU(cudaMemsetAsync(ss->sig, 0xff, (size_t)pl->nuniq * pl->npix * sizeof(float), st), "sigma preset");
    if (running && !ss->var_init) // the recursion of a trial starts at its first valid push: NaN = "not started" (also after a reset)
        SCU(cudaMemsetAsync(ss->var, 0xff, (size_t)pl->nuniq * pl->npix * sizeof(float), st), "running variance preset");
    for (int b = 0; b < npass; ++b) {
        StreamParams sp;
        sp.ring = ss->ring; sp.mu0 = ss->mu0; sp.partials = ss->partials;
        sp.top_row = ss->guard + base_slot + len - 1;
        sp.len = len;
        sp.i0 = b * c.CMAX;
        sp.C = std::min(c.CMAX, chunk_nt - sp.i0);
        sp.nslice = nslice;
        sp.slice0 = b * c.NSUPER;
        sp.mws = ss->mws; sp.aws = ss->aws; sp.sws = ss->sws;
        sp.snr_cube = cs; sp.toa_cube = ct; sp.t_offset = (int32_t)(lo & 0x7fffffff);
        sp.sig_out = (running && !c.INCR) ? ss->sig : nullptr;
        sp.dlt = ss->dlt; sp.rsig = ss->rsig; sp.dh = ss->dhist; sp.dh8 = ss->dh8;
        segment_bounds(pl, c, len, sp.i0, sp.C, sp.bound);
        void *args[] = {&sp};
        dim3 grid((pl->npix + 31) / 32, c.NSUPER);
        SCU(cudaLaunchKernel((const void *)ss->fn[variant], grid, dim3(c.threads()), args, c.smem, st), "k_stream launch");
        ++*launches;
    }
    if (ss->snr_cube && pl->nuniq < pl->ndm) {   // (the library's own cubes are read for canonical trials only)
        dim3 grid((unsigned)((cube_plane + 255) / 256), pl->ndm);
        k_cube_dups<<<grid, 256, 0, st>>>(ss->snr_cube, ss->toa_cube, ss->d_canon, cube_plane);
        SCU(cudaGetLastError(), "k_cube_dups launch");
        ++*launches;
    }
    if (running) {
        k_running<<<(pl->npix + 255) / 256, 256, 0, st>>>(cs, ct, ss->sig, ss->var, pl->d_k_of_u, pl->nuniq, pl->nw, pl->npix,
                                                          pl->run_alpha, ss->var_init ? 0 : 1, pl->run_snr, pl->run_arg);
        SCU(cudaGetLastError(), "k_running launch");
        ss->var_init = true;
        ++*launches;
    }
    if (pl->profiling && pl->ev[2]) cudaEventRecord(pl->ev[2], st);
    k_stream_finalize<<<(pl->npix + 255) / 256, 256, 0, st>>>(ss->partials, nslice, pl->npix, (int)(lo & 0x7fffffff), snr_map, argmax);
    SCU(cudaGetLastError(), "k_stream_finalize launch");
    ++*launches;
    return NSFRB_OK;
}

} // namespace nsfrb
