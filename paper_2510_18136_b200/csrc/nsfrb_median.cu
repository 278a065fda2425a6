// Per-(channel, pixel) median subtraction (first part; "Data is first median
// subtracted in each pixel"; reading R29 in DESIGN.md).  HBM-bound by contract: every element read once, written once.
//   k_median_reg<NT>  nt <= 32 (the paper's 25-sample chunks): one thread per series (lanes = adjacent pixels, so
//                     every row access is coalesced), the series in registers, Batcher's odd-even merge network
//                     specialised at compile time for the exact length and for the two middle outputs.
//   k_median_tile<P>  longer series: a [P pixels][nt] tile of order-preserving integer keys in shared memory, exact
//                     radix select of all P series at once (4 passes of 8 bits, shared-memory histograms split over
//                     32/P sub-histograms per series, one warp scans a series' 256 counters), the upper middle
//                     element by one more pass (warp per series), subtraction on the way out.
#include "nsfrb_internal.h"

#include <cstdlib>

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

constexpr int kTileThreads = 512;
constexpr int kHistWords = 32 * 256;   // [P][S][256] counters with P*S = 32: 32 KB whatever the tile shape

template <int P>
__global__ void __launch_bounds__(kTileThreads) k_median_tile(const float *in, float *out,   // may alias
                                                              float *__restrict__ med, int nt, long long npix,
                                                              int stride)
{
    constexpr int S = 32 / P;            // sub-histograms per series (lanes spread over them: fewer same-bin conflicts)
    extern __shared__ uint32_t smem_u32[];
    uint32_t *hist = smem_u32;           // [P][S][256]
    uint32_t *keys = smem_u32 + kHistWords;   // [P][stride], stride odd
    __shared__ uint32_t s_prefix[P];
    __shared__ int s_k[P];
    __shared__ float smed[P];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = kTileThreads / 32;
    const long long c = blockIdx.y, p0 = (long long)blockIdx.x * P;
    const int np = (int)min((long long)P, npix - p0);
    const float *src = in + c * nt * npix + p0;
    const int total = nt * P;
    // asynchronous 4-byte copies straight into the transposed tile: no register dependence, so a thread keeps all of
    // its loads in flight (rows of P pixels are neither 16-byte aligned nor a multiple of 16 bytes in general)
    {
        const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(keys);
        for (int idx = tid; idx < total; idx += kTileThreads) {
            const int t = idx / P, p = idx % P;
            if (p < np)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sbase + 4u * (uint32_t)(p * stride + t)),
                             "l"(src + (long long)t * npix + p)
                             : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    for (int i = tid; i < kHistWords; i += kTileThreads) hist[i] = 0;
    const int k1 = (nt - 1) >> 1, k2 = nt >> 1;
    if (tid < P) {
        s_prefix[tid] = 0;
        s_k[tid] = k1;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    // ---- exact order statistic k1 of every series: 4 passes of 8 bits, all warps over all series
    for (int pass = 0; pass < 4; ++pass) {
        const int shift = 24 - 8 * pass;
        // P >= 16 (short series): a warp per series; P <= 8 (long series): the whole CTA walks one series at a time.
        // Pass 0 also turns the float bits the copies delivered into order-preserving keys, in place.
        const int pstep = P >= 16 ? NW : 1, tstep = P >= 16 ? 32 : kTileThreads;
        for (int p = P >= 16 ? warp : 0; p < np; p += pstep) {
            uint32_t *row = keys + p * stride;
            uint32_t *hp = hist + ((p * S + (lane & (S - 1))) << 8);
            const uint32_t prefix = s_prefix[p];
            if (pass == 0) {
#pragma unroll 4
                for (int t = P >= 16 ? lane : tid; t < nt; t += tstep) {
                    const uint32_t key = ord_key(__uint_as_float(row[t]));
                    row[t] = key;
                    atomicAdd(hp + (key >> 24), 1u);
                }
            } else {
#pragma unroll 4
                for (int t = P >= 16 ? lane : tid; t < nt; t += tstep) {
                    const uint32_t key = row[t];
                    if (((key ^ prefix) >> (shift + 8)) == 0u) atomicAdd(hp + ((key >> shift) & 255u), 1u);
                }
            }
        }
        __syncthreads();
        for (int p = warp; p < np; p += NW) {      // lane l owns digits 8l..8l+7
            uint32_t cnt[8];
            uint32_t tot = 0;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                uint32_t v = 0;
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    uint32_t *h = &hist[((p * S + q) << 8) + 8 * lane + i];
                    v += *h;
                    *h = 0;
                }
                cnt[i] = v;
                tot += v;
            }
            uint32_t incl = tot;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t x = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += x;
            }
            const uint32_t excl = incl - tot, k = (uint32_t)s_k[p];
            if (excl <= k && k < incl) {
                uint32_t run = excl;
                int d = 0;
                bool found = false;
#pragma unroll
                for (int i = 0; i < 8; ++i)
                    if (!found) {
                        if (k < run + cnt[i]) {
                            found = true;
                            d = i;
                        } else
                            run += cnt[i];
                    }
                s_prefix[p] |= (uint32_t)(8 * lane + d) << shift;
                s_k[p] = (int)(k - run);
            }
        }
        __syncthreads();
    }
    // ---- even nt: the next order statistic (same value if it repeats, else the next key up); the median
    for (int p = warp; p < np; p += NW) {
        const uint32_t *row = keys + p * stride;
        const uint32_t prefix = s_prefix[p];
        uint32_t hi = prefix;
        if (k2 != k1) {
            int le = 0;
            uint32_t nxt = 0xffffffffu;
            for (int t = lane; t < nt; t += 32) {
                const uint32_t q = row[t];
                le += q <= prefix;
                nxt = q > prefix ? min(nxt, q) : nxt;
            }
            le = __reduce_add_sync(0xffffffffu, le);
            nxt = __reduce_min_sync(0xffffffffu, nxt);
            if (le <= k2) hi = nxt;
        }
        if (lane == 0) {
            const float m = middle(ord_val(prefix), ord_val(hi));
            smed[p] = m;
            if (med) med[c * npix + p0 + p] = m;
        }
    }
    __syncthreads();
    float *dst = out + c * nt * npix + p0;
    for (int idx = tid; idx < total; idx += kTileThreads) {
        const int t = idx / P, p = idx % P;
        if (p < np) dst[(long long)t * npix + p] = ord_val(keys[p * stride + t]) - smed[p];
    }
}

template <int NT>
cudaError_t launch_reg(const float *in, float *out, float *med, int nchan, long long npix, cudaStream_t st)
{
    const long long ns = (long long)nchan * npix;
    k_median_reg<NT><<<(unsigned)((ns + 255) / 256), 256, 0, st>>>(in, out, med, npix, ns);
    return cudaGetLastError();
}

template <int P>
cudaError_t launch_tile(const float *in, float *out, float *med, int nchan, int nt, long long npix, int stride,
                        cudaStream_t st)
{
    const size_t smem = ((size_t)P * stride + kHistWords) * sizeof(uint32_t);
    static size_t granted_dev[64] = {};   // only ever raised (another call may be using the kernel concurrently)
    int dev = 0;
    cudaGetDevice(&dev);
    size_t &granted = granted_dev[dev & 63];
    if (smem > 48 * 1024 && smem > granted) {
        cudaError_t e = cudaFuncSetAttribute(k_median_tile<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        granted = smem;
    }
    dim3 grid((unsigned)((npix + P - 1) / P), (unsigned)nchan);
    k_median_tile<P><<<grid, kTileThreads, smem, st>>>(in, out, med, nt, npix, stride);
    return cudaGetLastError();
}

} // namespace

int median_max_nt() { return ((200 - 32) * 1024 / 4 - 1) | 1; }

int median_tile_pixels(int nt)
{
    const int stride = nt | 1;
    int p = 32;
    if (const char *e = getenv("NSFRB_MEDIAN_P")) return atoi(e);
    while (p > 8 && (size_t)p * stride * 4 > (72 - 32) * 1024) p >>= 1;   // three CTAs per SM while rows stay >= 32 bytes
    while (p > 1 && (size_t)p * stride * 4 > (200 - 32) * 1024) p >>= 1;  // (32 KB of every CTA are the histograms)
    return p;
}

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
    const int stride = nt | 1;
    switch (median_tile_pixels(nt)) {
    case 32: return launch_tile<32>(in, out, med, nchan, nt, npix, stride, st);
    case 16: return launch_tile<16>(in, out, med, nchan, nt, npix, stride, st);
    case 8: return launch_tile<8>(in, out, med, nchan, nt, npix, stride, st);
    case 4: return launch_tile<4>(in, out, med, nchan, nt, npix, stride, st);
    case 2: return launch_tile<2>(in, out, med, nchan, nt, npix, stride, st);
    default: return launch_tile<1>(in, out, med, nchan, nt, npix, stride, st);
    }
}

} // namespace nsfrb
