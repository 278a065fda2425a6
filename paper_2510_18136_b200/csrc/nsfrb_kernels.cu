// sm_100a kernels of the NSFRB search hot path (steps a1..a8 of DESIGN.md):
//   k_transpose / k_push : cube or chunk [chan][time][pixel] -> workspace W[pixel][chan][time]
//                          (time-contiguous, per-channel baseline removed); a8 ring update
//   k_search             : dedispersion shift-and-sum (a2), mean/variance (a1, a3), prefix sum
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

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(kFull, v, o));
    return v;
}
__device__ __forceinline__ int warp_min_i(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(kFull, v, o));
    return v;
}
__device__ __forceinline__ int warp_max_i(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(kFull, v, o));
    return v;
}

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
                                                   int npix, int nchan, int nt, int pitch)
{
    __shared__ float tile[32][33];
    const int c = blockIdx.z;
    const int p0 = blockIdx.x * 32, t0 = blockIdx.y * 32;
    const size_t chan0 = (size_t)c * nt * (size_t)npix;
    {
        const int p = p0 + threadIdx.x;
        const float b = (p < npix) ? __ldg(cube + chan0 + p) : 0.f;
        for (int r = threadIdx.y; r < 32; r += 8) {
            const int t = t0 + r;
            if (t < nt && p < npix) tile[r][threadIdx.x] = __ldg(cube + chan0 + (size_t)t * npix + p) - b;
        }
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int p = p0 + r, t = t0 + threadIdx.x;
        if (t < nt && p < npix) W[((size_t)p * nchan + c) * (size_t)pitch + t] = tile[threadIdx.x][r];
    }
}

// chunk[c][i][p] -> W[p][c][(slot0 + i) mod L] - base[c][p]; the first push defines base.
__global__ void __launch_bounds__(256) k_push(const float *__restrict__ chunk, float *__restrict__ W,
                                              float *__restrict__ base, int npix, int nchan, int chunk_nt,
                                              int pitch, int ring_L, int slot0, int set_base)
{
    __shared__ float tile[32][33];
    const int c = blockIdx.y;
    const int p0 = blockIdx.x * 32;
    const size_t chan0 = (size_t)c * chunk_nt * (size_t)npix;
    const int pr = p0 + threadIdx.x;
    float b = 0.f;
    if (pr < npix) {
        b = set_base ? __ldg(chunk + chan0 + pr) : base[(size_t)c * npix + pr];
        if (set_base && threadIdx.y == 0) base[(size_t)c * npix + pr] = b;
    }
    for (int i0 = 0; i0 < chunk_nt; i0 += 32) {
        for (int r = threadIdx.y; r < 32; r += 8) {
            const int i = i0 + r;
            if (i < chunk_nt && pr < npix) tile[r][threadIdx.x] = __ldg(chunk + chan0 + (size_t)i * npix + pr) - b;
        }
        __syncthreads();
        for (int r = threadIdx.y; r < 32; r += 8) {
            const int p = p0 + r, i = i0 + threadIdx.x;
            if (i < chunk_nt && p < npix) {
                int slot = slot0 + i;
                if (slot >= ring_L) slot -= ring_L;
                W[((size_t)p * nchan + c) * (size_t)pitch + slot] = tile[threadIdx.x][r];
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------
// Search kernel.  One CTA = one pixel x one group of kSearchWarps DM trials x one batch of
// <= 32 widths.  Warp w owns trial u = g*kSearchWarps + w end to end; lanes run across time.
// The CTA sweeps time in blocks of kBlockLen dedispersed samples:
//   all warps : stage raw[c][t0 .. t0+kBlockLen+dmax_g) of the pixel in shared memory
//   each warp : D = shift-and-sum over channels (8 samples per lane, stride 32)
//               x = D - mu0 (mu0 = mean of the first block; the exact mean enters at the end)
//               s1 += x, s2 += x^2
//               P = running prefix of x (warp scans), stored in the warp's ring of H samples
//               for every width: m_j = max(m_j, P[e] - P[e-w_j]) over the block's ends e
// Validity is carried by infinities, not predicates: ring slots "before time 0" hold +inf and
// ends outside [e_min, T_k] are -inf in registers, so an undefined cell evaluates to -inf.
// At the end: delta = s1/T (mu = mu0+delta), var = s2/T - delta^2, and because
// sum_{window}(D-mu) = sum_{window}(D-mu0) - w*delta, max_t B_j = m_j - w_j*delta exactly.
// ------------------------------------------------------------------------------------------
template <int NWARP>
__global__ void __launch_bounds__(NWARP * 32, 1) k_search(const SearchParams P)
{
    extern __shared__ __align__(16) float smem[];
    const int nchan = P.nchan, RS = P.RS, H = P.H;
    float *raw = smem;                          // [nchan][RS]
    float *rings = raw + (size_t)nchan * RS;    // [NWARP][H]
    int *sw = reinterpret_cast<int *>(rings + (size_t)NWARP * H); // [32] widths of this batch
    float *red_s = reinterpret_cast<float *>(sw + kWidthBatch);   // [NWARP]
    int *red_i = reinterpret_cast<int *>(red_s + NWARP);          // [NWARP][4] k, j, u, -
    float *red_f = reinterpret_cast<float *>(red_i + 4 * NWARP);  // [NWARP][2] mu, sigma
    int *grp = reinterpret_cast<int *>(red_f + 2 * NWARP);        // [2] dmax_g, dmin_g

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int slices = P.n_groups * P.n_wb;
    const int p = blockIdx.x / slices;
    const int sl = blockIdx.x - p * slices;
    const int g = sl / P.n_wb, wb = sl - g * P.n_wb;
    const int u = g * NWARP + warp;
    const int nwb = min(kWidthBatch, P.nw - wb * kWidthBatch);

    const int dmax_k = (u < P.nuniq) ? __ldg(P.dmax_u + u) : 0;
    const bool has = (u < P.nuniq) && (P.len - dmax_k >= 1); // a trial with no valid sample yet has no cell
    const int T_k = has ? P.len - dmax_k : 0;
    const int emin_k = P.raw_end_min - dmax_k + 1; // ends e >= emin_k are evaluated (S5)
    const int32_t *dk = P.delays_u + (size_t)(has ? u : 0) * nchan;
    float *ring = rings + (size_t)warp * H;

    if (threadIdx.x < kWidthBatch)
        sw[threadIdx.x] = threadIdx.x < nwb ? __ldg(P.widths + wb * kWidthBatch + threadIdx.x) : 1;
    if (warp == 0) {
        int dmx = 0, dmn = 0x7fffffff;
        for (int i = lane; i < NWARP; i += 32) {
            const int uu = g * NWARP + i;
            if (uu < P.nuniq) {
                const int d = __ldg(P.dmax_u + uu);
                dmx = max(dmx, d);
                dmn = min(dmn, d);
            }
        }
        dmx = warp_max_i(dmx);
        dmn = warp_min_i(dmn);
        if (lane == 0) { grp[0] = dmx; grp[1] = dmn; }
    }
    for (int i = lane; i < H; i += 32) ring[i] = (i == 0) ? 0.f : CUDART_INF_F;
    __syncthreads();
    const int dmax_g = grp[0];
    const int T_g = P.len - grp[1]; // longest series of the group
    const int rows = kBlockLen + dmax_g;
    const float *Wp = P.W + (size_t)p * nchan * (size_t)P.pitch;

    float m[kWidthBatch];
#pragma unroll
    for (int j = 0; j < kWidthBatch; ++j) m[j] = -CUDART_INF_F;
    float mu0 = 0.f, s1 = 0.f, s2 = 0.f, carry = 0.f;
    int te = 1; // (t0 + 1) mod H

    for (int t0 = 0; t0 < T_g; t0 += kBlockLen) {
        // ---- stage the raw block: relative samples [t0, t0+rows) of every channel
        __syncthreads();
        for (int c = warp; c < nchan; c += NWARP) {
            const float *src = Wp + (size_t)c * P.pitch;
            float *dst = raw + (size_t)c * RS;
            for (int i = lane; i < rows; i += 32) {
                const int r = t0 + i;
                float v = 0.f;
                if (r < P.len) {
                    int slot = P.origin + r;
                    if (slot >= P.ring_L) slot -= P.ring_L;
                    v = __ldg(src + slot);
                }
                dst[i] = v;
            }
        }
        __syncthreads();
        if (!has || t0 >= T_k) continue;

        // ---- a2: shift-and-sum
        float acc[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[i] = 0.f;
        for (int c = 0; c < nchan; ++c) {
            const float *r = raw + (size_t)c * RS + __ldg(dk + c) + lane;
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[i] += r[32 * i];
        }
        if (t0 == 0) {
            float s = 0.f;
#pragma unroll
            for (int i = 0; i < 8; ++i) s += (lane + 32 * i < T_k) ? acc[i] : 0.f;
            s = warp_sum(s);
            mu0 = s / (float)min(kBlockLen, T_k);
        }
        // ---- a3 partial sums, a4 prefix
        float Pe[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int t = t0 + lane + 32 * i;
            float x = (t < T_k) ? acc[i] - mu0 : 0.f;
            s1 += x;
            s2 = fmaf(x, x, s2);
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const float y = __shfl_up_sync(kFull, x, o);
                if (lane >= o) x += y;
            }
            x += carry;
            carry = __shfl_sync(kFull, x, 31);
            Pe[i] = x; // = P[t+1]
        }
        {
            int a = te + lane;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                int pos = a + 32 * i;
                if (pos >= H) pos -= H;
                ring[pos] = Pe[i];
            }
        }
        __syncwarp();
        // ---- a5: boxcars ending in this block
        if (t0 + kBlockLen >= emin_k) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int e = t0 + 1 + lane + 32 * i;
                if (e > T_k || e < emin_k) Pe[i] = -CUDART_INF_F;
            }
#pragma unroll
            for (int j = 0; j < kWidthBatch; ++j) {
                if (j < nwb) {
                    int q = te - sw[j]; // ring slot of the first start
                    if (q < 0) q += H;
                    float mj = m[j];
                    if (q + kBlockLen <= H) {
                        const float *b = ring + q + lane;
#pragma unroll
                        for (int i = 0; i < 8; ++i) mj = fmaxf(mj, Pe[i] - b[32 * i]);
                    } else {
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            unsigned a = (unsigned)(q + lane + 32 * i);
                            a = min(a, a - (unsigned)H);
                            mj = fmaxf(mj, Pe[i] - ring[a]);
                        }
                    }
                    m[j] = mj;
                }
            }
        }
        te += kBlockLen;
        if (te >= H) te -= H;
        __syncwarp();
    }

    // ---- a6 (per trial): exact mean / variance, normalise, best width
    float bs = -CUDART_INF_F;
    int bj = -1;
    float mu = 0.f, sigma = 0.f;
    if (has) {
        const float S1 = warp_sum(s1), S2 = warp_sum(s2);
        const float invT = 1.f / (float)T_k;
        const float delta = S1 * invT;
        const float var = fmaxf(fmaf(-delta, delta, S2 * invT), 0.f);
        sigma = sqrtf(var);
        mu = mu0 + delta;
#pragma unroll
        for (int j = 0; j < kWidthBatch; ++j) {
            const float mj = warp_max(m[j]);
            if (j < nwb && mj > -CUDART_INF_F) {
                const float w = (float)sw[j];
                const float B = fmaf(-w, delta, mj);
                const float S = sigma > 0.f ? B / (sigma * sqrtf(w)) : 0.f;
                if (bj < 0 || S > bs) { bs = S; bj = j; }
            }
        }
    }
    if (lane == 0) {
        red_s[warp] = bs;
        red_i[4 * warp + 0] = (has && bj >= 0) ? __ldg(P.k_of_u + u) : -1;
        red_i[4 * warp + 1] = bj < 0 ? -1 : wb * kWidthBatch + bj;
        red_i[4 * warp + 2] = u;
        red_f[2 * warp + 0] = mu;
        red_f[2 * warp + 1] = sigma;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        Partial out;
        out.snr = -CUDART_INF_F; out.k = -1; out.j = -1; out.blk = -1; out.mu = 0.f; out.sigma = 0.f; out.u = -1; out.pad = 0;
        for (int w = 0; w < NWARP; ++w) {
            if (better(red_s[w], red_i[4 * w], red_i[4 * w + 1], out.snr, out.k, out.j)) {
                out.snr = red_s[w]; out.k = red_i[4 * w]; out.j = red_i[4 * w + 1]; out.u = red_i[4 * w + 2];
                out.mu = red_f[2 * w]; out.sigma = red_f[2 * w + 1];
            }
        }
        P.partials[(size_t)p * slices + sl] = out;
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
// host-side launchers
// ------------------------------------------------------------------------------------------
size_t search_smem_bytes(int nchan, int RS, int H)
{
    size_t n = (size_t)nchan * RS + (size_t)kSearchWarps * H; // floats
    n += kWidthBatch + kSearchWarps + 4 * kSearchWarps + 2 * kSearchWarps + 2;
    return n * sizeof(float) + 16;
}

size_t final_smem_bytes(int nt) { return ((size_t)nt + 2) * sizeof(float); }

cudaError_t configure_kernels(size_t search_smem, size_t final_smem)
{
    cudaError_t e = cudaFuncSetAttribute(k_search<kSearchWarps>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)search_smem);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_finalize, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)final_smem);
}

cudaError_t launch_transpose(const float *cube, float *W, int npix, int nchan, int nt, int pitch, cudaStream_t st)
{
    dim3 grid((npix + 31) / 32, (nt + 31) / 32, nchan), block(32, 8);
    k_transpose<<<grid, block, 0, st>>>(cube, W, npix, nchan, nt, pitch);
    return cudaGetLastError();
}

cudaError_t launch_push(const float *chunk, float *W, float *base, int npix, int nchan, int chunk_nt, int pitch,
                        int ring_L, int slot0, int set_base, cudaStream_t st)
{
    dim3 grid((npix + 31) / 32, nchan), block(32, 8);
    k_push<<<grid, block, 0, st>>>(chunk, W, base, npix, nchan, chunk_nt, pitch, ring_L, slot0, set_base);
    return cudaGetLastError();
}

cudaError_t launch_search(const SearchParams &p, size_t smem_bytes, cudaStream_t st)
{
    const long long blocks = (long long)p.npix * p.n_groups * p.n_wb;
    if (blocks <= 0 || blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    k_search<kSearchWarps><<<(unsigned)blocks, kSearchWarps * 32, smem_bytes, st>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_finalize(const FinalParams &p, size_t smem_bytes, cudaStream_t st)
{
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
