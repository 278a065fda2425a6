// sm_100a kernels of the NSFRB search hot path (steps a1..a8 of DESIGN.md):
//   k_transpose          : cube [chan][time][pixel] -> workspace W[pixel][chan][time]
//                          (time-contiguous, per-channel baseline removed)
//   k_search             : (nsfrb_search.cu) dedispersion (a2), mean/variance (a1, a3), prefix sum
//                          (a4), boxcar + peak over time (a5), S/N + reduction over (DM, width)
//                          of one DM group (a6, first half)
//   k_finalize           : reduction over groups, arg-max time by rescanning the winning
//                          series (a6, second half)
//   k_compact            : threshold + warp-aggregated candidate compaction (a7)
// Definitions: include/nsfrb.h.  No code is shared with oracle/.
#include <math_constants.h>

#include "nsfrb_internal.h"

namespace nsfrb {

namespace {

constexpr unsigned kFull = 0xffffffffu;


// (snr, k, j) ordering of O6: larger snr wins; exact ties go to the smaller k, then smaller j.
__device__ __forceinline__ bool better(float s, int k, int j, float bs, int bk, int bj)
{
    if (k < 0) return false;
    if (bk < 0) return true;
    if (s != bs) return s > bs;
    if (k != bk) return k < bk;
    return j < bj;
}

} // namespace

// ------------------------------------------------------------------------------------------
// a8 / layout change.  W[p][c][t] = I[c][t][p] - I[c][0][p]
// The per-(channel, pixel) constant cancels exactly in D_k - mu_k; removing it keeps float32
// sums at the scale of the fluctuations instead of the sky level.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_transpose(const float *__restrict__ cube, float *__restrict__ W,
                                                   int npix, int nchan, int nt, int pitch, int p_begin, int p_end)
{
    // 64 pixels x 64 samples per CTA: 256-byte runs on both the read (pixel-contiguous) and the write
    // (time-contiguous) side; 65-float rows keep both shared-memory phases conflict-free or 2-way
    __shared__ float tile[64][65];
    const int c = blockIdx.z;
    const int p0 = p_begin + blockIdx.x * 64, t0 = blockIdx.y * 64;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const size_t chan0 = (size_t)c * nt * (size_t)npix;
    {
        const int pa = p0 + lane, pb = p0 + 32 + lane;
        const float ba = (pa < p_end) ? __ldg(cube + chan0 + pa) : 0.f;
        const float bb = (pb < p_end) ? __ldg(cube + chan0 + pb) : 0.f;
#pragma unroll 4
        for (int r = warp; r < 64; r += 8) {
            const int t = t0 + r;
            if (t < nt) {
                const float *row = cube + chan0 + (size_t)t * npix;
                if (pa < p_end) tile[r][lane] = __ldcs(row + pa) - ba;
                if (pb < p_end) tile[r][32 + lane] = __ldcs(row + pb) - bb;
            }
        }
    }
    __syncthreads();
#pragma unroll 4
    for (int r = warp; r < 64; r += 8) {
        const int p = p0 + r;
        if (p < p_end) {
            float *dst = W + ((size_t)(p - p_begin) * nchan + c) * (size_t)pitch + t0;
            if (t0 + lane < nt) dst[lane] = tile[lane][r];
            if (t0 + 32 + lane < nt) dst[32 + lane] = tile[32 + lane][r];
        }
    }
}

// ------------------------------------------------------------------------------------------
// a6 second half: best slice of the pixel, then the arg-max time by recomputing the winning
// series over the range of starts that can hold it, with the mean/sigma the search found.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_finalize(const FinalParams F)
{
    extern __shared__ __align__(16) float fs[]; // [n+1] prefix, then scratch
    __shared__ Partial best;
    __shared__ float sc_f[256];
    __shared__ int sc_i[256];
    const int p = blockIdx.x;
    const int tid = threadIdx.x;
    if (tid == 0) {
        Partial b;
        b.snr = -CUDART_INF_F; b.k = -1; b.j = -1; b.blk = -1; b.mu = 0.f; b.sigma = 0.f; b.u = -1; b.pad = 0;
        const Partial *pp = F.partials + (size_t)p * F.slices;
        for (int s = 0; s < F.slices; ++s) {
            const Partial c = pp[s];
            if (better(c.snr, c.k, c.j, b.snr, b.k, b.j)) b = c;
        }
        best = b;
    }
    __syncthreads();
    const Partial b = best;
    if (b.k < 0) {
        if (tid == 0) {
            F.snr_map[p] = -CUDART_INF_F;
            F.argmax[p] = -1; F.argmax[(size_t)F.npix + p] = -1; F.argmax[2 * (size_t)F.npix + p] = -1;
        }
        return;
    }
    const int w = __ldg(F.widths + b.j);
    const int dmax = __ldg(F.dmax_u + b.u);
    const int T = F.len - dmax;
    const int emin = F.raw_end_min - dmax + 1;
    const int e_lo = max(w, emin);
    const int ta = e_lo - w;  // first start
    const int n = T - ta;     // samples [ta, T)
    const int32_t *dk = F.delays_u + (size_t)b.u * F.nchan;
    const float *Wp = F.W + (size_t)p * F.nchan * (size_t)F.pitch;

    // x[i] = D[ta+i] - mu, staged at fs[i+1]
    for (int i = tid; i < n; i += 256) {
        float s = 0.f;
        for (int c = 0; c < F.nchan; ++c) {
            int slot = F.origin + ta + i + __ldg(dk + c);
            if (slot >= F.ring_L) slot -= F.ring_L;
            s += __ldg(Wp + (size_t)c * F.pitch + slot);
        }
        fs[i + 1] = s - b.mu;
    }
    if (tid == 0) fs[0] = 0.f;
    __syncthreads();
    // block-wide inclusive scan of fs[1..n]: odd-length chunk per thread (conflict-free)
    const int ch = ((n + 255) / 256) | 1;
    const int a0 = 1 + tid * ch, a1 = min(a0 + ch, n + 1);
    float tot = 0.f;
    for (int i = a0; i < a1; ++i) tot += fs[i];
    sc_f[tid] = tot;
    __syncthreads();
    if (tid < 32) {
        // scan of the 256 chunk totals by one warp, 8 per lane
        float v[8], run = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) { v[i] = sc_f[tid * 8 + i]; run += v[i]; }
        float incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const float y = __shfl_up_sync(kFull, incl, o);
            if (tid >= o) incl += y;
        }
        float ex = incl - run;
#pragma unroll
        for (int i = 0; i < 8; ++i) { sc_f[tid * 8 + i] = ex; ex += v[i]; }
    }
    __syncthreads();
    {
        float run = sc_f[tid];
        for (int i = a0; i < a1; ++i) { run += fs[i]; fs[i] = run; }
    }
    __syncthreads();
    // arg-max over starts i in [0, n-w]: B = P[i+w] - P[i], smallest i on ties
    float bv = -CUDART_INF_F;
    int bi = 0x7fffffff;
    for (int i = tid; i <= n - w; i += 256) {
        const float B = fs[i + w] - fs[i];
        if (B > bv) { bv = B; bi = i; }
    }
    sc_f[tid] = bv; sc_i[tid] = bi;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o) {
            const float ov = sc_f[tid + o]; const int oi = sc_i[tid + o];
            if (ov > sc_f[tid] || (ov == sc_f[tid] && oi < sc_i[tid])) { sc_f[tid] = ov; sc_i[tid] = oi; }
        }
        __syncthreads();
    }
    if (tid == 0) {
        const float B = sc_f[0];
        const float S = b.sigma > 0.f ? B / (b.sigma * sqrtf((float)w)) : 0.f;
        F.snr_map[p] = S;
        F.argmax[p] = b.k;
        F.argmax[(size_t)F.npix + p] = __ldg(F.j_of_used + b.j);
        F.argmax[2 * (size_t)F.npix + p] = (int32_t)(((uint32_t)F.t_offset + (uint32_t)(ta + sc_i[0])) & 0x7fffffffu);
    }
}

// The same for short series (nt <= 2048): one WARP per pixel, 8 pixels per CTA, no block-wide barrier -- the
// block-per-pixel version spends its time in __syncthreads when a series is only a few hundred samples (C4).
__global__ void __launch_bounds__(256) k_finalize_warp(const FinalParams F)
{
    extern __shared__ __align__(16) float fsw[]; // [8][pitchw]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int p = blockIdx.x * 8 + warp;
    if (p >= F.npix) return;
    const int pitchw = F.len + 3;
    float *fs = fsw + (size_t)warp * pitchw;
    // best slice of the pixel (lane 0), broadcast
    Partial b;
    b.snr = -CUDART_INF_F; b.k = -1; b.j = -1; b.blk = -1; b.mu = 0.f; b.sigma = 0.f; b.u = -1; b.pad = 0;
    if (lane == 0) {
        const Partial *pp = F.partials + (size_t)p * F.slices;
        for (int s = 0; s < F.slices; ++s) {
            const Partial c = pp[s];
            if (better(c.snr, c.k, c.j, b.snr, b.k, b.j)) b = c;
        }
    }
    b.k = __shfl_sync(kFull, b.k, 0); b.j = __shfl_sync(kFull, b.j, 0); b.u = __shfl_sync(kFull, b.u, 0);
    b.mu = __shfl_sync(kFull, b.mu, 0); b.sigma = __shfl_sync(kFull, b.sigma, 0);
    if (b.k < 0) {
        if (lane == 0) {
            F.snr_map[p] = -CUDART_INF_F;
            F.argmax[p] = -1; F.argmax[(size_t)F.npix + p] = -1; F.argmax[2 * (size_t)F.npix + p] = -1;
        }
        return;
    }
    const int w = __ldg(F.widths + b.j);
    const int dmax = __ldg(F.dmax_u + b.u);
    const int T = F.len - dmax;
    const int emin = F.raw_end_min - dmax + 1;
    const int ta = max(w, emin) - w; // first start
    const int n = T - ta;            // samples [ta, T)
    const int32_t *dk = F.delays_u + (size_t)b.u * F.nchan;
    const float *Wp = F.W + (size_t)p * F.nchan * (size_t)F.pitch;
    for (int i = lane; i < n; i += 32) {
        float s = 0.f;
        for (int c = 0; c < F.nchan; ++c) {
            int slot = F.origin + ta + i + __ldg(dk + c);
            if (slot >= F.ring_L) slot -= F.ring_L;
            s += __ldg(Wp + (size_t)c * F.pitch + slot);
        }
        fs[i + 1] = s - b.mu;
    }
    if (lane == 0) fs[0] = 0.f;
    __syncwarp();
    // inclusive scan of fs[1..n]: odd-length chunk per lane (conflict-free), one warp scan of the chunk totals
    const int ch = ((n + 31) / 32) | 1;
    const int a0 = 1 + lane * ch, a1 = min(a0 + ch, n + 1);
    float tot = 0.f;
    for (int i = a0; i < a1; ++i) tot += fs[i];
    float incl = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const float y = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += y;
    }
    {
        float run = incl - tot;
        for (int i = a0; i < a1; ++i) { run += fs[i]; fs[i] = run; }
    }
    __syncwarp();
    float bv = -CUDART_INF_F;
    int bi = 0x7fffffff;
    for (int i = lane; i <= n - w; i += 32) {
        const float B = fs[i + w] - fs[i];
        if (B > bv) { bv = B; bi = i; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(kFull, bv, o);
        const int oi = __shfl_xor_sync(kFull, bi, o);
        if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    if (lane == 0) {
        const float S = b.sigma > 0.f ? bv / (b.sigma * sqrtf((float)w)) : 0.f;
        F.snr_map[p] = S;
        F.argmax[p] = b.k;
        F.argmax[(size_t)F.npix + p] = __ldg(F.j_of_used + b.j);
        F.argmax[2 * (size_t)F.npix + p] = (int32_t)(((uint32_t)F.t_offset + (uint32_t)(ta + bi)) & 0x7fffffffu);
    }
}

// ------------------------------------------------------------------------------------------
// a7: snr > threshold -> candidate list, one atomicAdd per warp.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_compact(const float *__restrict__ snr_map, const int32_t *__restrict__ argmax,
                                                 int npix, float threshold, nsfrb_cand *cands, uint32_t cap,
                                                 uint32_t *ncands)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    float s = -CUDART_INF_F;
    if (p < npix) s = snr_map[p];
    const bool hit = (p < npix) && (s > threshold);
    const unsigned mask = __ballot_sync(kFull, hit);
    if (mask == 0) return;
    const int leader = __ffs(mask) - 1;
    uint32_t base = 0;
    if (lane == leader) base = atomicAdd(ncands, (uint32_t)__popc(mask));
    base = __shfl_sync(kFull, base, leader);
    if (hit) {
        const uint32_t idx = base + (uint32_t)__popc(mask & ((1u << lane) - 1u));
        if (idx < cap) {
            nsfrb_cand c;
            c.pixel = p;
            c.dm_idx = argmax[p];
            c.width_idx = argmax[(size_t)npix + p];
            c.t = argmax[2 * (size_t)npix + p];
            c.snr = s;
            cands[idx] = c;
        }
    }
}

// ------------------------------------------------------------------------------------------
// NEXT 2: time binning out[c][u][p] = sum_{i<factor} in[c][u*factor+i][p]  (reading R24).
// One thread owns one output vector (1 or 4 pixels) and walks `factor` input rows: coalesced, every input
// byte read once -- HBM-bound by construction.
// ------------------------------------------------------------------------------------------
template <typename V>
__global__ void __launch_bounds__(256) k_bin(const V *__restrict__ in, V *__restrict__ out, int nt, int nb, long long npv,
                                             int factor)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npv) return;
    const int c = blockIdx.z;
    for (int u = blockIdx.y; u < nb; u += gridDim.y) {
        const V *src = in + ((size_t)c * nt + (size_t)u * factor) * npv + p;
        V acc = __ldcs(src);
        for (int i = 1; i < factor; ++i) {
            const V v = __ldcs(src + (size_t)i * npv);
            if constexpr (sizeof(V) == 16) { acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w; }
            else acc += v;
        }
        out[((size_t)c * nb + u) * npv + p] = acc;
    }
}

cudaError_t launch_bin(const float *in, float *out, int nchan, int nt, long long npix, int factor, cudaStream_t st)
{
    const int nb = nt / factor;
    if (nb < 1) return cudaSuccess;
    const bool v4 = (npix % 4 == 0) && (((reinterpret_cast<uintptr_t>(in) | reinterpret_cast<uintptr_t>(out)) & 15u) == 0);
    const long long npv = v4 ? npix / 4 : npix;
    dim3 grid((unsigned)((npv + 255) / 256), (unsigned)(nb < 65535 ? nb : 65535), (unsigned)nchan);
    if (v4) k_bin<float4><<<grid, 256, 0, st>>>(reinterpret_cast<const float4 *>(in), reinterpret_cast<float4 *>(out), nt, nb, npv, factor);
    else k_bin<float><<<grid, 256, 0, st>>>(in, out, nt, nb, npv, factor);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// host-side launchers
// ------------------------------------------------------------------------------------------
size_t final_smem_bytes(int nt) { return ((size_t)nt + 2) * sizeof(float); }

cudaError_t launch_transpose(const float *cube, float *W, int npix, int nchan, int nt, int pitch, int p_begin, int p_count,
                             cudaStream_t st)
{
    if (p_count <= 0) return cudaSuccess;
    dim3 grid((p_count + 63) / 64, (nt + 63) / 64, nchan), block(256);
    k_transpose<<<grid, block, 0, st>>>(cube, W, npix, nchan, nt, pitch, p_begin, p_begin + p_count);
    return cudaGetLastError();
}

cudaError_t launch_finalize(const FinalParams &p, size_t smem_bytes, cudaStream_t st)
{
    static size_t granted[64] = {0}, granted_w[64] = {0}; // per-device function attributes shared by all plans: only ever raise them
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (p.len <= 2048) { // short series: one warp per pixel
        const size_t smw = 8 * ((size_t)p.len + 3) * sizeof(float);
        if (dev >= 0 && dev < 64 && smw > granted_w[dev]) {
            e = cudaFuncSetAttribute(k_finalize_warp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smw);
            if (e != cudaSuccess) return e;
            granted_w[dev] = smw;
        }
        k_finalize_warp<<<(p.npix + 7) / 8, 256, smw, st>>>(p);
        return cudaGetLastError();
    }
    if (dev >= 0 && dev < 64 && smem_bytes > granted[dev]) {
        e = cudaFuncSetAttribute(k_finalize, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return e;
        granted[dev] = smem_bytes;
    }
    k_finalize<<<p.npix, 256, smem_bytes, st>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_compact(const float *snr_map, const int32_t *argmax, int npix, float threshold, nsfrb_cand *cands,
                           uint32_t cap, uint32_t *ncands, cudaStream_t st)
{
    k_compact<<<(npix + 255) / 256, 256, 0, st>>>(snr_map, argmax, npix, threshold, cands, cap, ncands);
    return cudaGetLastError();
}

} // namespace nsfrb
