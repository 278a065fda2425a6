// Post-search candidate selection (second part): PSF percentile mask,
// the N highest-S/N per-pixel candidates, PSF-mask sidelobe clustering with a weighted mean S/N per centre.
// Readings R25..R28 in DESIGN.md.  Two kernels:
//   k_psf_mask  one CTA: exact order statistics of the PSF by a 4-pass radix select on order-preserving keys,
//               linear interpolation in float64 (no contraction), then the strict comparison of every element.
//   k_cluster   one launch: every CTA selects the N best (S/N, pixel) keys of its slice of the map by N rounds of
//               "largest key below the previous winner"; the last CTA to finish (ticket) merges the per-CTA lists
//               the same way, then one thread per centre walks the N candidates in rank order.
#include <mutex>

#include "nsfrb_internal.h"

namespace nsfrb {
namespace {

constexpr int kSelThreads = 1024;
constexpr int kCluThreads = 256;
constexpr int kMaxTop = 32;

// float -> uint32 that sorts like the float (-inf < ... < -0 < +0 < ... < +inf)
__device__ __forceinline__ uint32_t ord_key(float f)
{
    const uint32_t b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float ord_val(uint32_t k)
{
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

__global__ void __launch_bounds__(kSelThreads) k_psf_mask(const float *__restrict__ psf, long long n, long long lo,
                                                          double frac, uint8_t *__restrict__ mask,
                                                          double *__restrict__ value)
{
    __shared__ unsigned int hist[256];
    __shared__ uint32_t s_prefix;
    __shared__ unsigned long long s_rank, s_le;
    __shared__ uint32_t s_next;
    __shared__ double s_thr;
    const int tid = threadIdx.x;
    uint32_t prefix = 0;            // bits of the rank-lo key found so far
    unsigned long long rank = (unsigned long long)lo;
    for (int pass = 0; pass < 4; ++pass) {
        const int shift = 24 - 8 * pass;
        const uint32_t himask = pass == 0 ? 0u : (0xffffffffu << (shift + 8));
        if (tid < 256) hist[tid] = 0;
        __syncthreads();
        for (long long i = tid; i < n; i += kSelThreads) {
            const uint32_t k = ord_key(psf[i]);
            if ((k & himask) == prefix) atomicAdd(&hist[(k >> shift) & 255u], 1u);
        }
        __syncthreads();
        if (tid == 0) {
            unsigned long long r = rank;
            int b = 0;
            for (; b < 255; ++b) {
                if (r < hist[b]) break;
                r -= hist[b];
            }
            s_prefix = prefix | ((uint32_t)b << shift);
            s_rank = r;
        }
        __syncthreads();
        prefix = s_prefix;
        rank = s_rank;
        __syncthreads();
    }
    // the order statistic above it: the same value if it is repeated, else the smallest larger key
    if (tid == 0) {
        s_le = 0;
        s_next = 0xffffffffu;
    }
    __syncthreads();
    unsigned long long le = 0;
    uint32_t nxt = 0xffffffffu;
    for (long long i = tid; i < n; i += kSelThreads) {
        const uint32_t k = ord_key(psf[i]);
        if (k <= prefix) ++le;
        else nxt = min(nxt, k);
    }
    atomicAdd(&s_le, le);
    atomicMin(&s_next, nxt);
    __syncthreads();
    if (tid == 0) {
        const double vlo = (double)ord_val(prefix);
        double vhi = vlo;
        if (lo + 1 < n && s_le < (unsigned long long)lo + 2) vhi = (double)ord_val(s_next);
        s_thr = __dadd_rn(vlo, __dmul_rn(frac, __dsub_rn(vhi, vlo)));
        if (value) *value = s_thr;
    }
    __syncthreads();
    const double thr = s_thr;
    for (long long i = tid; i < n; i += kSelThreads) mask[i] = (double)psf[i] > thr ? 1 : 0;
}

// (S/N, pixel) -> one 64-bit key: larger S/N first, then the smaller pixel.  0 = "no candidate".
__device__ __forceinline__ unsigned long long cand_key(float s, uint32_t p)
{
    return ((unsigned long long)ord_key(s) << 32) | (unsigned long long)(0xffffffffu - p);
}

__device__ __forceinline__ unsigned long long block_max(unsigned long long v, unsigned long long *red)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long x = __shfl_xor_sync(0xffffffffu, v, o);
        v = x > v ? x : v;
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();                     // red[] may still be read from the previous round
    if (l == 0) red[w] = v;
    __syncthreads();
    v = l < kCluThreads / 32 ? red[l] : 0ull;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) {
        const unsigned long long x = __shfl_xor_sync(0xffffffffu, v, o);
        v = x > v ? x : v;
    }
    return __shfl_sync(0xffffffffu, v, 0);
}

struct ClusterParams {
    const float *snr_map;
    const int32_t *argmax;   // [3][npix]
    const float *psf;
    const uint8_t *mask;
    unsigned long long *ws;  // [gridDim.x][topn] keys
    unsigned int *ticket;
    nsfrb_cand *top;
    double *wsnr;
    int32_t *members;
    int32_t *result;         // {n_found, best}
    int npix, nx, mh, mw, topn, slice;
    float threshold;
};

__global__ void __launch_bounds__(kCluThreads) k_cluster(const ClusterParams P)
{
    __shared__ unsigned long long red[kCluThreads / 32];
    __shared__ unsigned long long top[kMaxTop];
    __shared__ double s_w[kMaxTop];
    __shared__ bool s_last;
    const int tid = threadIdx.x;
    // ---- the N best of this CTA's slice
    const int p0 = blockIdx.x * P.slice, p1 = min(P.npix, p0 + P.slice);
    unsigned long long bound = ~0ull;
    for (int r = 0; r < P.topn; ++r) {
        unsigned long long best = 0;
        if (bound != 0)
            for (int p = p0 + tid; p < p1; p += kCluThreads) {
                const float s = __ldg(P.snr_map + p);
                if (s > P.threshold) {
                    const unsigned long long k = cand_key(s, (uint32_t)p);
                    if (k < bound && k > best) best = k;
                }
            }
        bound = bound != 0 ? block_max(best, red) : 0ull;
        if (tid == 0) P.ws[(size_t)blockIdx.x * P.topn + r] = bound;
    }
    // ---- last CTA merges
    __threadfence();
    if (tid == 0) s_last = atomicAdd(P.ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int nkeys = (int)gridDim.x * P.topn;
    bound = ~0ull;
    for (int r = 0; r < P.topn; ++r) {
        unsigned long long best = 0;
        if (bound != 0)
            for (int i = tid; i < nkeys; i += kCluThreads) {
                const unsigned long long k = __ldcg(P.ws + i);
                if (k < bound && k > best) best = k;
            }
        bound = bound != 0 ? block_max(best, red) : 0ull;
        if (tid == 0) top[r] = bound;
    }
    __syncthreads();
    int nfound = 0;
    while (nfound < P.topn && top[nfound] != 0) ++nfound;
    // ---- one thread per centre: members inside the mask, weighted mean in rank order (float64, no contraction)
    if (tid < P.topn) {
        nsfrb_cand c = {-1, -1, -1, -1, 0.f};
        double wm = 0.0;
        int cnt = 0;
        if (tid < nfound) {
            const int cy = P.mh / 2, cx = P.mw / 2;
            const int pi = (int)(0xffffffffu - (uint32_t)(top[tid] & 0xffffffffu));
            const int xi = pi % P.nx, yi = pi / P.nx;
            double num = 0.0, den = 0.0;
            for (int j = 0; j < nfound; ++j) {
                const int pj = (int)(0xffffffffu - (uint32_t)(top[j] & 0xffffffffu));
                const int mx = cx + (pj % P.nx - xi), my = cy + (pj / P.nx - yi);
                const bool inside = mx >= 0 && mx < P.mw && my >= 0 && my < P.mh;
                float w;
                if (j == tid) w = P.psf[(size_t)cy * P.mw + cx];
                else if (inside && P.mask[(size_t)my * P.mw + mx]) w = P.psf[(size_t)my * P.mw + mx];
                else continue;
                const double s = (double)ord_val((uint32_t)(top[j] >> 32));
                num = __dadd_rn(num, __dmul_rn((double)w, s));
                den = __dadd_rn(den, (double)w);
                ++cnt;
            }
            wm = __ddiv_rn(num, den);
            c.pixel = pi;
            c.dm_idx = P.argmax[pi];
            c.width_idx = P.argmax[(size_t)P.npix + pi];
            c.t = P.argmax[2 * (size_t)P.npix + pi];
            c.snr = ord_val((uint32_t)(top[tid] >> 32));
        }
        P.top[tid] = c;
        P.wsnr[tid] = wm;
        P.members[tid] = cnt;
        s_w[tid] = wm;
    }
    __syncthreads();
    if (tid == 0) {
        int best = -1;
        for (int i = 0; i < nfound; ++i)
            if (best < 0 || s_w[i] > s_w[best]) best = i;
        P.result[0] = nfound;
        P.result[1] = best;
        *P.ticket = 0;          // ready for the next call on this stream
    }
}

} // namespace

cudaError_t launch_psf_mask(const float *psf, long long n, long long lo, double frac, uint8_t *mask, double *value,
                            cudaStream_t st)
{
    k_psf_mask<<<1, kSelThreads, 0, st>>>(psf, n, lo, frac, mask, value);
    return cudaGetLastError();
}

int cluster_max_top() { return kMaxTop; }

int cluster_grid(int npix)
{
    // at least 2048 pixels per CTA, at most one CTA per SM of a B200
    const int g = (npix + 2047) / 2048;
    return g < 1 ? 1 : (g > 148 ? 148 : g);
}

cudaError_t launch_cluster(const float *snr_map, const int32_t *argmax, int npix, int nx, float threshold,
                           const float *psf, const uint8_t *mask, int mh, int mw, int topn, void *ws,
                           unsigned int *ticket, nsfrb_cand *top, double *wsnr, int32_t *members, int32_t *result,
                           cudaStream_t st)
{
    ClusterParams P;
    const int grid = cluster_grid(npix);
    P.snr_map = snr_map;
    P.argmax = argmax;
    P.psf = psf;
    P.mask = mask;
    P.ws = static_cast<unsigned long long *>(ws);
    P.ticket = ticket;
    P.top = top;
    P.wsnr = wsnr;
    P.members = members;
    P.result = result;
    P.npix = npix;
    P.nx = nx;
    P.mh = mh;
    P.mw = mw;
    P.topn = topn;
    P.slice = (npix + grid - 1) / grid;
    P.threshold = threshold;
    k_cluster<<<grid, kCluThreads, 0, st>>>(P);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// nsfrb_cluster_static: the same kernel for callers that may not allocate (CUDA graph capture, serving loops, harnesses
// that forbid cudaMalloc).  Its workspace -- the ticket (first 256 bytes) and the per-CTA key lists,
// kStaticCtas x kMaxTop keys -- is this file-scope array: 38 144 bytes that every GPU which loads the library holds
// until exit.  All calls share it, so two calls that overlap on one GPU (different streams) race; it keeps the last
// call's contents: the key lists are fully rewritten by every launch before they are read, the ticket is cleared on the
// caller's stream before every launch.
// In host code `g_cluster_scratch` is only a stand-in for the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int kStaticCtas = 148;                 // cluster_grid never launches more CTAs
constexpr int kStaticMaxNpix = 1 << 24;          // stated limit of the entry point (a 4096 x 4096 map)
constexpr int kStaticWords = 32 + kStaticCtas * kMaxTop; // 64-bit words: 256-byte header + keys
static __device__ __align__(256) unsigned long long g_cluster_scratch[kStaticWords];

constexpr int kMaxDevices = 64;
unsigned long long *g_scratch_addr[kMaxDevices] = {nullptr};
std::mutex g_scratch_mutex;

// device address of the scratch on the current device (looked up once per device)
cudaError_t cluster_static_scratch(unsigned long long **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        unsigned long long *ptr = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void **>(&ptr), g_cluster_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

} // namespace

int cluster_static_max_npix() { return kStaticMaxNpix; }

// No cudaMalloc/cudaFree and no allocating library call on this path: symbol lookup (first call per device), one
// 256-byte cudaMemsetAsync, one kernel launch.
cudaError_t launch_cluster_static(const float *snr_map, const int32_t *argmax, int npix, int nx, float threshold,
                                  const float *psf, const uint8_t *mask, int mh, int mw, int topn, nsfrb_cand *top,
                                  double *wsnr, int32_t *members, int32_t *result, cudaStream_t st)
{
    if (npix < 1 || npix > kStaticMaxNpix || topn < 1 || topn > kMaxTop || cluster_grid(npix) > kStaticCtas)
        return cudaErrorInvalidValue; // (the C entry point reports these with their own messages first)
    unsigned long long *scratch = nullptr;
    cudaError_t e = cluster_static_scratch(&scratch);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(scratch, 0, 256, st); // the ticket must start at zero whatever an earlier call left behind
    if (e != cudaSuccess) return e;
    return launch_cluster(snr_map, argmax, npix, nx, threshold, psf, mask, mh, mw, topn, scratch + 32,
                          reinterpret_cast<unsigned int *>(scratch), top, wsnr, members, result, st);
}

} // namespace nsfrb
