// Per-(channel, pixel) median subtraction (first part; "Data is first median
// subtracted in each pixel"; reading R29 in DESIGN.md).  HBM-bound by contract: every element read once, written once.
//   k_median_reg<NT>  nt <= 32 (the paper's 25-sample chunks): one thread per series (lanes = adjacent pixels, so
//                     every row access is coalesced), the series in registers, Batcher's odd-even merge network
//                     specialised at compile time for the exact length and for the two middle outputs.
//   k_median_stream   longer series (<= 65 535 samples): lanes = adjacent pixels again, nothing but lane-private 8-bit
//                     histograms on chip; three streaming reads of the series (histogram, candidates, subtraction)
//                     and one write for noise-like data; exact for any data (more histogram passes when a bucket
//                     stays crowded).
#include "nsfrb_internal.h"

namespace nsfrb {
namespace {

__device__ __forceinline__ uint32_t ord_key(float f)
{
    const uint32_t b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float ord_val(uint32_t k)
{
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}
// mean of the two middle elements in float64, rounded once (equal elements give the element back)
__device__ __forceinline__ float middle(float lo, float hi)
{
    return __double2float_rn(__dmul_rn(0.5, __dadd_rn((double)lo, (double)hi)));
}

__host__ __device__ constexpr int pow2_ceil(int n) { return n <= 1 ? 1 : 2 * pow2_ceil((n + 1) / 2); }

// Batcher's odd-even merge sort for N = 2^k >= NT inputs (iterative form), as a comparator list.  The network is in
// standard form (minimum to the lower index), so with +inf in the places NT..N-1 every comparator whose upper index
// is >= NT does nothing and is left out.
struct NetList {
    int n;
    int lo[192], hi[192];
};
__host__ __device__ constexpr NetList make_net(int nt)
{
    NetList r{};
    const int N = pow2_ceil(nt);
    for (int pp = 1; pp < N; pp <<= 1)
        for (int k = pp; k >= 1; k >>= 1)
            for (int j = k % pp; j <= N - 1 - k; j += 2 * k)
                for (int i = 0; i <= (k - 1 < N - j - k - 1 ? k - 1 : N - j - k - 1); ++i)
                    if ((i + j) / (2 * pp) == (i + j + k) / (2 * pp) && i + j + k < nt) {
                        r.lo[r.n] = i + j;
                        r.hi[r.n] = i + j + k;
                        ++r.n;
                    }
    return r;
}
template <int NT>
struct Net {
    static constexpr NetList value = make_net(NT);
};

template <int I>
struct IC {
    static constexpr int v = I;
};
template <int LO, int HI, class F>
__device__ __forceinline__ void sfor(F &&f)      // f(IC<LO>) ... f(IC<HI-1>), every index a constant expression
{
    if constexpr (HI - LO == 1)
        f(IC<LO>{});
    else if constexpr (HI - LO > 1) {
        constexpr int M = (LO + HI) / 2;
        sfor<LO, M>(f);
        sfor<M, HI>(f);
    }
}

// NT = the exact series length: every index below is a compile-time constant after unrolling, so the series lives in
// registers, comparators that would touch the (virtual, +inf) padding are dropped and the ones that cannot reach the
// two middle outputs are removed by the compiler.
template <int NT>
__global__ void __launch_bounds__(256) k_median_reg(const float *in, float *out,   // may alias (in place)
                                                    float *__restrict__ med, long long npix, long long nseries)
{
    __shared__ float keep[NT][256];    // the unsorted series for the subtraction (a second register copy would
    float x[NT];                       // halve the occupancy; a second global read misses L1 most of the time)
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nseries) return;
    const long long c = s / npix, p = s - c * npix;
    const float *src = in + c * NT * npix + p;
    {
        const float *q = src;          // running pointers: one 64-bit add per row instead of a 64-bit multiply
#pragma unroll
        for (int i = 0; i < NT; ++i) {
            x[i] = *q;
            keep[i][threadIdx.x] = x[i];
            q += npix;
        }
    }
    // the comparators as compile-time constants: x[] never leaves the registers
    sfor<0, Net<NT>::value.n>([&](auto e) {
        constexpr int a = Net<NT>::value.lo[decltype(e)::v], b = Net<NT>::value.hi[decltype(e)::v];
        const float u = x[a], w = x[b];
        x[a] = fminf(u, w);
        x[b] = fmaxf(u, w);
    });
    const float m = middle(x[(NT - 1) / 2], x[NT / 2]);
    if (med) med[s] = m;
    float *dst = out + c * NT * npix + p;
#pragma unroll
    for (int i = 0; i < NT; ++i) {
        *dst = keep[i][threadIdx.x] - m;
        dst += npix;
    }
}

// ---- long series, streaming form: lanes = adjacent pixels, one warp = 32 series of one channel.  Nothing but the
// histograms is kept on chip, so every row access is a coalesced 128-byte line whatever nt and npix are.
//   pass H (one read of the series): lane-private 8-bit histograms of the keys that match the prefix found so far
//                                    ([256 bins][32 lanes] 16-bit counters: no atomics, no bank conflicts);
//                                    repeated on the next 8 bits only while some series still has > kCap matching keys
//   pass C (one read):               the <= kCap matching keys of every series go to shared memory (over the histograms),
//                                    together with the smallest key above the bucket; exact selection among them
//   pass W (one read, one write):    out = x - median
// Noise-like data needs H, C, W: three reads and one write (2x the minimal traffic), all of it streaming.
constexpr int kMsWarps = 4;
constexpr int kCap = 128;                       // candidate keys per series: [kCap][32] uint32 = the 16 KB of the histograms
constexpr int kMsSmemPerWarp = 256 * 32 * 2;    // bytes

// f(x, t) for t = 0..nt-1 over one series (row stride npix), with the loads of the next kMsU rows already requested
// while the current kMsU are processed (two register batches: up to 64 rows in flight per lane).
constexpr int kMsU = 16;
template <class F>
__device__ __forceinline__ void for_rows(const float *src, int nt, long long npix, F &&f)
{
    float a[kMsU], b[kMsU];
    const int nb = nt / kMsU;
    const float *q = src;              // running pointer: rows are requested strictly in order
    auto load = [&](float (&x)[kMsU], int) {
#pragma unroll
        for (int i = 0; i < kMsU; ++i) {
            x[i] = *q;
            q += npix;
        }
    };
    auto run = [&](const float (&x)[kMsU], int t0) {
#pragma unroll
        for (int i = 0; i < kMsU; ++i) f(x[i], t0 + i);
    };
    if (nb > 0) load(a, 0);
    for (int ib = 0; ib < nb; ib += 2) {
        if (ib + 1 < nb) load(b, (ib + 1) * kMsU);
        run(a, ib * kMsU);
        if (ib + 1 < nb) {
            if (ib + 2 < nb) load(a, (ib + 2) * kMsU);
            run(b, (ib + 1) * kMsU);
        }
    }
    for (int t = nb * kMsU; t < nt; ++t) f(src[(long long)t * npix], t);
}

__global__ void __launch_bounds__(kMsWarps * 32, 3) k_median_stream(const float *in, float *out,   // may alias
                                                                 float *__restrict__ med, int nt, long long npix,
                                                                 int blocks_per_chan, long long nwork)
{
    extern __shared__ uint32_t smem_u32[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long work = (long long)blockIdx.x * kMsWarps + warp;    // (channel, block of 32 pixels)
    if (work >= nwork) return;
    uint16_t *hist = reinterpret_cast<uint16_t *>(smem_u32 + warp * (kMsSmemPerWarp / 4));   // [256][32]
    uint32_t *cand = smem_u32 + warp * (kMsSmemPerWarp / 4);                                 // [kCap][32], same bytes
    const long long c = work / blocks_per_chan, p = (work - c * blocks_per_chan) * 32 + lane;
    const bool live = p < npix;
    const float *src = in + c * nt * npix + (live ? p : 0);
    const int k1 = (nt - 1) >> 1, k2 = nt >> 1;
    uint32_t prefix = 0;
    int nbits = 0;                 // leading key bits already fixed
    int k = k1;                    // rank of the wanted key among the keys that match the prefix
    int count = live ? nt : 0;     // how many keys match the prefix
    // ---- pass H, as often as needed
    while (__any_sync(0xffffffffu, count > kCap && nbits < 32)) {
        for (int i = lane; i < 256 * 32 / 2; i += 32) reinterpret_cast<uint32_t *>(hist)[i] = 0;
        __syncwarp();
        const int shift = 24 - nbits;
        const bool all = nbits == 0;
        const bool on = live && nbits < 32;
        if (on)
            for_rows(src, nt, npix, [&](float x, int) {
                const uint32_t key = ord_key(x);
                if (all || ((key ^ prefix) >> (shift + 8)) == 0u) ++hist[((key >> shift) & 255u) * 32 + lane];
            });
        __syncwarp();
        if (on) {                  // the bin that holds rank k
            int run = 0, b = 0, h = 0;
            for (; b < 256; ++b) {
                h = hist[b * 32 + lane];
                if (k < run + h) break;
                run += h;
            }
            prefix |= (uint32_t)b << shift;
            k -= run;
            count = h;
        }
        nbits += 8;                // (uniform: every series of the warp moves on together)
        __syncwarp();
    }
    // ---- pass C: candidates and the smallest key above the bucket
    const bool undecided = live && nbits < 32;
    uint32_t key1 = prefix, key2 = prefix;
    if (__any_sync(0xffffffffu, undecided) || k2 != k1) {
        const uint32_t hi_bound = nbits >= 32 ? prefix : (prefix | (0xffffffffu >> nbits));   // largest key of the bucket
        uint32_t nxt = 0xffffffffu;
        int n = 0;
        if (live)
            for_rows(src, nt, npix, [&](float x, int) {
                const uint32_t key = ord_key(x);
                if (key > hi_bound) nxt = min(nxt, key);
                else if (undecided && (nbits == 0 || ((key ^ prefix) >> (32 - nbits)) == 0u)) cand[(n++) * 32 + lane] = key;
            });
        if (undecided) {           // exact selection among the n <= kCap candidates: the remaining bits, one at a time
            const int r = k;
            uint32_t pfx = prefix;
            for (int b = 31 - nbits; b >= 0; --b) {
                int cnt = 0;
                for (int i = 0; i < n; ++i) cnt += ((cand[i * 32 + lane] ^ pfx) >> b) == 0u;
                if (k >= cnt) {
                    k -= cnt;
                    pfx |= 1u << b;
                }
            }
            key1 = pfx;
            int le = 0;
            uint32_t up = 0xffffffffu;
            for (int i = 0; i < n; ++i) {
                const uint32_t q = cand[i * 32 + lane];
                le += q <= key1;
                up = q > key1 ? min(up, q) : up;
            }
            key2 = r + 1 < le ? key1 : (up != 0xffffffffu ? up : nxt);
        } else {                   // all 32 bits fixed: `count` keys equal key1, the wanted one is the k-th of them
            key2 = k + 1 < count ? key1 : nxt;
        }
    }
    if (!live) return;
    const float m = k2 != k1 ? middle(ord_val(key1), ord_val(key2)) : ord_val(key1);
    if (med) med[c * npix + p] = m;
    // ---- pass W
    float *dst = out + c * nt * npix + p;
    for_rows(src, nt, npix, [&](float x, int t) { dst[(long long)t * npix] = x - m; });
}

cudaError_t launch_stream(const float *in, float *out, float *med, int nchan, int nt, long long npix, cudaStream_t st)
{
    const size_t smem = (size_t)kMsWarps * kMsSmemPerWarp;
    static bool granted_dev[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (!granted_dev[dev & 63]) {
        cudaError_t e = cudaFuncSetAttribute(k_median_stream, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        granted_dev[dev & 63] = true;
    }
    const long long bpc = (npix + 31) / 32, nwork = bpc * nchan;
    k_median_stream<<<(unsigned)((nwork + kMsWarps - 1) / kMsWarps), kMsWarps * 32, smem, st>>>(in, out, med, nt, npix, (int)bpc, nwork);
    return cudaGetLastError();
}

template <int NT>
cudaError_t launch_reg(const float *in, float *out, float *med, int nchan, long long npix, cudaStream_t st)
{
    const long long ns = (long long)nchan * npix;
    k_median_reg<NT><<<(unsigned)((ns + 255) / 256), 256, 0, st>>>(in, out, med, npix, ns);
    return cudaGetLastError();
}

} // namespace

int median_max_nt() { return 65535; }   // 16-bit histogram counters of k_median_stream

cudaError_t launch_median(const float *in, float *out, float *med, int nchan, int nt, long long npix, cudaStream_t st)
{
    switch (nt) {
#define NSFRB_MEDIAN_REG(n) case n: return launch_reg<n>(in, out, med, nchan, npix, st);
        NSFRB_MEDIAN_REG(1) NSFRB_MEDIAN_REG(2) NSFRB_MEDIAN_REG(3) NSFRB_MEDIAN_REG(4) NSFRB_MEDIAN_REG(5)
        NSFRB_MEDIAN_REG(6) NSFRB_MEDIAN_REG(7) NSFRB_MEDIAN_REG(8) NSFRB_MEDIAN_REG(9) NSFRB_MEDIAN_REG(10)
        NSFRB_MEDIAN_REG(11) NSFRB_MEDIAN_REG(12) NSFRB_MEDIAN_REG(13) NSFRB_MEDIAN_REG(14) NSFRB_MEDIAN_REG(15)
        NSFRB_MEDIAN_REG(16) NSFRB_MEDIAN_REG(17) NSFRB_MEDIAN_REG(18) NSFRB_MEDIAN_REG(19) NSFRB_MEDIAN_REG(20)
        NSFRB_MEDIAN_REG(21) NSFRB_MEDIAN_REG(22) NSFRB_MEDIAN_REG(23) NSFRB_MEDIAN_REG(24) NSFRB_MEDIAN_REG(25)
        NSFRB_MEDIAN_REG(26) NSFRB_MEDIAN_REG(27) NSFRB_MEDIAN_REG(28) NSFRB_MEDIAN_REG(29) NSFRB_MEDIAN_REG(30)
        NSFRB_MEDIAN_REG(31) NSFRB_MEDIAN_REG(32)
#undef NSFRB_MEDIAN_REG
    default: break;
    }
    return launch_stream(in, out, med, nchan, nt, npix, st);
}

} // namespace nsfrb
