// k_search: the hot kernel of the NSFRB search (steps a1..a6 of DESIGN.md) for sm_100a.
//
// One CTA = one pixel x one group of kSearchWarps (16) DM trials x one batch of <= 32 widths.
// The CTA sweeps the pixel's time axis in blocks of kBlockLen (256) dedispersed samples; the
// dedispersed series, its prefix sum and every boxcar live in shared memory / registers only.
//
//   cp.async      raw[c][t0 .. t0+256+dmax_g) of the pixel for block b+1 is fetched from the
//                 time-contiguous workspace while block b is searched (the raw tile is only read
//                 by phase 1, so one buffer is enough)
//   phase 1 (CTA) differential dedispersion (a2): thread (half h, sample tl) walks 8 consecutive
//                 DM trials; the first is the plain sum over channels, every next one adds
//                 raw[c][t+d'] - raw[c][t+d] for the channels whose delay changed (plan-time change
//                 lists, 2-10x fewer operands than nchan).  D goes to a padded staging tile.
//   phase 2 (warp w = trial w): 8 consecutive samples per lane
//                 x = D - mu0, s1 += x, s2 += x^2                      (a1, a3; exact mean at the end)
//                 prefix P: 8 serial adds + one warp scan per 8 samples  (a4)
//                 P -> the warp's ring of H samples, row minima of P per 32 samples
//                 widths <= 16: boxcars straight from a 24-sample register window      (a5)
//                 widths  > 16: exact branch-and-bound.  Lane j bounds width j for the block by
//                   max(P over valid ends) - min(P over the 9 rows holding its starts); only if that
//                   can beat the running maximum M_j is the block evaluated from the ring
//                   (LDS + FADD + FMNMX per cell, one CREDUX.MAX.F32 per block).  Every cell of a
//                   skipped block is <= the bound <= M_j, so max_t is unchanged.
// Validity is carried by infinities: ring slots before time 0 hold +inf (P[0] = 0 sits in slot H-1),
// ends outside [e_min, T_k] are -inf, so an undefined cell evaluates to -inf without predicates.
// End of series: delta = s1/T (mu = mu0+delta), var = s2/T - delta^2, max_t B_j = M_j - w_j*delta
// exactly, S_j = B_j/(sigma sqrt(w_j)); lanes hold one width each, a shuffle arg-max picks (S, j).
#include <math_constants.h>

#include "nsfrb_internal.h"

namespace nsfrb {

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr int NW = kSearchWarps;
constexpr int LB = kBlockLen;
constexpr int SS = kStageStride;
constexpr int kSmallW = 16; // widths served from registers

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
// CREDUX.MAX.F32: warp-wide float max in one instruction (sm_100a)
__device__ __forceinline__ float warp_max(float v)
{
    float r;
    asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
    return r;
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
__device__ __forceinline__ void cp_async16(float *dst, const float *src, int src_bytes)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async4(float *dst, const float *src, int src_bytes)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(d), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// raw[c][i] = W[p][c][slot(t0+i)] for i < rows4, zero beyond the valid samples
__device__ __forceinline__ void issue_raw(const SearchParams &P, const float *Wp, float *raw, int t0, int rows4, int warp,
                                          int lane, bool aligned)
{
    for (int c = warp; c < P.nchan; c += NW) {
        const float *src = Wp + (size_t)c * P.pitch;
        float *dst = raw + (size_t)c * P.RS;
        if (aligned) {
            for (int i = lane * 4; i < rows4; i += 128) {
                const int r = t0 + i;
                const int nvalid = max(0, min(4, P.len - r));
                int slot = P.origin + r;
                if (slot >= P.ring_L) slot -= P.ring_L;
                if (nvalid == 0) slot = 0;
                cp_async16(dst + i, src + slot, nvalid * 4);
            }
        } else {
            for (int i = lane; i < rows4; i += 32) {
                const int r = t0 + i;
                const bool ok = r < P.len;
                int slot = P.origin + r;
                if (slot >= P.ring_L) slot -= P.ring_L;
                if (!ok) slot = 0;
                cp_async4(dst + i, src + slot, ok ? 4 : 0);
            }
        }
    }
    cp_async_commit();
}

// (snr, k, j) ordering of the definition: larger snr wins; exact ties go to the smaller k, then j.
__device__ __forceinline__ bool better(float s, int k, int j, float bs, int bk, int bj)
{
    if (k < 0) return false;
    if (bk < 0) return true;
    if (s != bs) return s > bs;
    if (k != bk) return k < bk;
    return j < bj;
}

} // namespace

__global__ void __launch_bounds__(NW * 32, 1) k_search(const SearchParams P)
{
    extern __shared__ __align__(16) float smem[];
    const int nchan = P.nchan, RS = P.RS, H = P.H, NR = P.H >> 5;
    float *raw = smem;                                  // [nchan][RS] (+4 pad)
    float *stage = raw + (size_t)nchan * RS + 4;        // [NW][SS]   padded: index t + 4*(t>>5)
    float *rings = stage + NW * SS;                     // [NW][H]    P[t+1] at slot t mod H
    float *rmins = rings + (size_t)NW * H;              // [NW][NR]   min of P over each 32-slot row
    int *tab = reinterpret_cast<int *>(rmins + NW * NR); // [tab_cap] dedispersion change lists of the group
    int *sw = tab + P.tab_cap;                          // [32] widths of this batch (0 = unused lane)
    int *jsm = sw + kWidthBatch;                        // [20] width value (1..16) -> lane, -1 if absent
    float *red_s = reinterpret_cast<float *>(jsm + 20); // [NW]
    int *red_i = reinterpret_cast<int *>(red_s + NW);   // [NW][4] k, j, u, -
    float *red_f = reinterpret_cast<float *>(red_i + 4 * NW); // [NW][2] mu, sigma
    int *grp = reinterpret_cast<int *>(red_f + 2 * NW); // [4] dmax_g, dmin_g

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int slices = P.n_groups * P.n_wb;
    const int p = blockIdx.x / slices;
    const int sl = blockIdx.x - p * slices;
    const int g = sl / P.n_wb, wb = sl - g * P.n_wb;
    const int u = g * NW + warp;
    const int nwb = min(kWidthBatch, P.nw - wb * kWidthBatch);

    const int dmax_k = (u < P.nuniq) ? __ldg(P.dmax_u + u) : 0;
    const bool has = (u < P.nuniq) && (P.len - dmax_k >= 1); // a trial with no valid sample yet has no cell
    const int T_k = has ? P.len - dmax_k : 0;
    const int emin_k = P.raw_end_min - dmax_k + 1; // ends e >= emin_k are evaluated (streaming rule S5)
    float *ring = rings + (size_t)warp * H;
    float *rmin = rmins + warp * NR;

    // ---- per-CTA setup
    {
        const int off = __ldg(P.dd_off + g), glen = __ldg(P.dd_off + g + 1) - off;
        for (int i = tid; i < glen; i += NW * 32) tab[i] = __ldg(P.dd_tab + off + i);
    }
    if (tid < kWidthBatch) sw[tid] = tid < nwb ? __ldg(P.widths + wb * kWidthBatch + tid) : 0;
    if (tid < 20) jsm[tid] = -1;
    if (warp == 0) {
        int dmx = 0, dmn = 0x7fffffff;
        for (int i = lane; i < NW; i += 32) {
            const int uu = g * NW + i;
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
    for (int i = lane; i < H; i += 32) ring[i] = (i == H - 1) ? 0.f : CUDART_INF_F; // P[0] = 0 at slot -1
    for (int i = lane; i < NR; i += 32) rmin[i] = (i == NR - 1) ? 0.f : CUDART_INF_F;
    __syncthreads();
    if (tid < nwb && sw[tid] <= kSmallW) jsm[sw[tid]] = tid;
    __syncthreads();
    unsigned smask = 0;
#pragma unroll
    for (int w = 1; w <= kSmallW; ++w) smask |= (jsm[w] >= 0 ? 1u : 0u) << w;
    const int wl = sw[lane];                 // this lane's width
    const bool is_large = wl > kSmallW;      // lanes >= nwb hold 0
    const bool any_large = __any_sync(kFull, is_large);
    int rr = ((-wl) >> 5) + NR;              // ring row of the first start of block 0 (floor division)
    if (rr >= NR || rr < 0) rr = 0;          // unused lanes

    const int dmax_g = grp[0];
    const int T_g = P.len - grp[1]; // longest series of the group
    const int rows4 = (LB + dmax_g + 3) & ~3;
    const float *Wp = P.W + (size_t)p * nchan * (size_t)P.pitch;
    const bool aligned = ((P.origin & 3) == 0) && (((P.ring_L & 3) == 0) || P.origin + P.len <= P.ring_L);

    float M = -CUDART_INF_F; // lane j: running max_t of the width-j boxcar (relative to mu0)
    float ms[kSmallW];
#pragma unroll
    for (int w = 0; w < kSmallW; ++w) ms[w] = -CUDART_INF_F;
    float mu0 = 0.f, s1 = 0.f, s2 = 0.f, carry = 0.f;
    int tpos = 0; // t0 mod H

    if (T_g > 0) issue_raw(P, Wp, raw, 0, rows4, warp, lane, aligned);

    for (int t0 = 0; t0 < T_g; t0 += LB) {
        cp_async_wait_all();
        __syncthreads(); // raw(b) landed; every warp is done with stage(b-1)

        // ---- phase 1: differential dedispersion of the block, all 16 trials
        {
            const int h = tid >> 8, tl = tid & (LB - 1);
            int pos = tab[h];
            const int nser = tab[pos];
            pos += 4;
            const float *rt = raw + tl;
            float *so = stage + (h * 8) * SS + tl + 4 * (tl >> 5);
            float acc = 0.f;
            for (int s = 0; s < nser; ++s) {
                const int n = tab[pos], type = tab[pos + 1];
                pos += 4;
                if (type == 0) { // plain sum over channels
                    acc = 0.f;
                    int c = 0;
                    for (; c + 4 <= n; c += 4) {
                        const int4 o = *reinterpret_cast<const int4 *>(tab + pos + c);
                        acc += (rt[o.x] + rt[o.y]) + (rt[o.z] + rt[o.w]);
                    }
                    for (; c < n; ++c) acc += rt[tab[pos + c]];
                    pos += (n + 3) & ~3;
                } else { // n groups of 4 (new, old) pairs
                    for (int q = 0; q < n; ++q) {
                        const int4 o0 = *reinterpret_cast<const int4 *>(tab + pos);
                        const int4 o1 = *reinterpret_cast<const int4 *>(tab + pos + 4);
                        acc += ((rt[o0.x] - rt[o0.y]) + (rt[o0.z] - rt[o0.w])) +
                               ((rt[o1.x] - rt[o1.y]) + (rt[o1.z] - rt[o1.w]));
                        pos += 8;
                    }
                }
                so[s * SS] = acc;
            }
        }
        __syncthreads(); // stage(b) complete; the raw tile is free again
        if (t0 + LB < T_g) issue_raw(P, Wp, raw, t0 + LB, rows4, warp, lane, aligned);

        // ---- phase 2: this warp's trial
        if (has && t0 < T_k) {
            float p8[8];
            {
                const float4 *sp = reinterpret_cast<const float4 *>(stage + warp * SS + 8 * lane + 4 * (lane >> 2));
                const float4 xa = sp[0], xb = sp[1];
                p8[0] = xa.x; p8[1] = xa.y; p8[2] = xa.z; p8[3] = xa.w;
                p8[4] = xb.x; p8[5] = xb.y; p8[6] = xb.z; p8[7] = xb.w;
            }
            const int tb = t0 + 8 * lane;
            const int nv = T_k - tb; // sample i of this lane is valid iff i < nv
            if (t0 == 0) {
                float s = 0.f;
#pragma unroll
                for (int i = 0; i < 8; ++i) s += (i < nv) ? p8[i] : 0.f;
                mu0 = warp_sum(s) / (float)min(LB, T_k);
            }
            float run = 0.f;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float x = (i < nv) ? p8[i] - mu0 : 0.f;
                s1 += x;
                s2 = fmaf(x, x, s2);
                run += x;
                p8[i] = run;
            }
            float incl = run;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const float y = __shfl_up_sync(kFull, incl, o);
                if (lane >= o) incl += y;
            }
            float excl = __shfl_up_sync(kFull, incl, 1);
            if (lane == 0) excl = 0.f;
            const float base = carry + excl;
#pragma unroll
            for (int i = 0; i < 8; ++i) p8[i] += base; // P[t+1], t = tb + i
            carry = __shfl_sync(kFull, p8[7], 31);

            int sb = tpos + 8 * lane; // ring slot of sample tb (8 | H, so the 8 slots never straddle the wrap)
            if (sb >= H) sb -= H;
            {
                float4 *rp = reinterpret_cast<float4 *>(ring + sb);
                rp[0] = make_float4(p8[0], p8[1], p8[2], p8[3]);
                rp[1] = make_float4(p8[4], p8[5], p8[6], p8[7]);
                float lmin = fminf(fminf(fminf(p8[0], p8[1]), fminf(p8[2], p8[3])),
                                   fminf(fminf(p8[4], p8[5]), fminf(p8[6], p8[7])));
                lmin = fminf(lmin, __shfl_xor_sync(kFull, lmin, 1));
                lmin = fminf(lmin, __shfl_xor_sync(kFull, lmin, 2));
                if ((lane & 3) == 0) rmin[sb >> 5] = lmin;
            }
            __syncwarp();

            if (t0 + LB >= emin_k) { // the block holds ends that are evaluated
                // ---- widths <= 16 from registers
                if (smask) {
                    float E[8], Wn[24];
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        E[i] = (i < nv && tb + i + 1 >= emin_k) ? p8[i] : -CUDART_INF_F;
                        Wn[16 + i] = p8[i];
                    }
                    int s2b = sb - 16, s1b = sb - 8;
                    if (s2b < 0) s2b += H;
                    if (s1b < 0) s1b += H;
                    {
                        const float4 *w2 = reinterpret_cast<const float4 *>(ring + s2b);
                        const float4 *w1 = reinterpret_cast<const float4 *>(ring + s1b);
                        const float4 a = w2[0], b = w2[1], c = w1[0], d = w1[1];
                        Wn[0] = a.x; Wn[1] = a.y; Wn[2] = a.z; Wn[3] = a.w; Wn[4] = b.x; Wn[5] = b.y; Wn[6] = b.z; Wn[7] = b.w;
                        Wn[8] = c.x; Wn[9] = c.y; Wn[10] = c.z; Wn[11] = c.w; Wn[12] = d.x; Wn[13] = d.y; Wn[14] = d.z; Wn[15] = d.w;
                    }
#pragma unroll
                    for (int w = 1; w <= kSmallW; ++w) {
                        if (smask & (1u << w)) {
                            float m = ms[w - 1];
#pragma unroll
                            for (int i = 0; i < 8; ++i) m = fmaxf(m, E[i] - Wn[16 + i - w]);
                            ms[w - 1] = m;
                        }
                    }
                }
                // ---- widths > 16: bound, then evaluate only the blocks that can raise the maximum
                if (any_large) {
                    float Pe[8], emx = -CUDART_INF_F;
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        int pos = tpos + lane + 32 * i;
                        if (pos >= H) pos -= H;
                        const int e = t0 + lane + 32 * i + 1;
                        const float v = (e <= T_k && e >= emin_k) ? ring[pos] : -CUDART_INF_F;
                        Pe[i] = v;
                        emx = fmaxf(emx, v);
                    }
                    const float Emax = warp_max(emx);
                    bool surv = false;
                    if (is_large) {
                        float mn = CUDART_INF_F;
                        int r = rr;
#pragma unroll
                        for (int q = 0; q < 9; ++q) {
                            mn = fminf(mn, rmin[r]);
                            if (++r == NR) r = 0;
                        }
                        surv = (Emax - mn) > M;
                    }
                    unsigned mask = __ballot_sync(kFull, surv);
                    while (mask) {
                        const int j = __ffs(mask) - 1;
                        mask &= mask - 1;
                        int q = tpos - sw[j]; // ring slot of the start that belongs to end slot tpos
                        if (q < 0) q += H;
                        float v = -CUDART_INF_F;
                        if (q + LB <= H) {
                            const float *b = ring + q + lane;
#pragma unroll
                            for (int i = 0; i < 8; ++i) v = fmaxf(v, Pe[i] - b[32 * i]);
                        } else {
#pragma unroll
                            for (int i = 0; i < 8; ++i) {
                                unsigned a = (unsigned)(q + lane + 32 * i);
                                a = min(a, a - (unsigned)H);
                                v = fmaxf(v, Pe[i] - ring[a]);
                            }
                        }
                        v = warp_max(v);
                        if (lane == j) M = fmaxf(M, v);
                    }
                }
            }
            __syncwarp();
        }
        tpos += LB;
        if (tpos >= H) tpos -= H;
        rr += LB / 32;
        if (rr >= NR) rr -= NR;
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
        for (int w = 1; w <= kSmallW; ++w) {
            if (smask & (1u << w)) {
                const float v = warp_max(ms[w - 1]);
                if (lane == jsm[w]) M = v;
            }
        }
        float S = -CUDART_INF_F;
        int jj = 0x7fffffff;
        if (lane < nwb && M > -CUDART_INF_F) {
            const float w = (float)wl;
            const float B = fmaf(-w, delta, M);
            S = sigma > 0.f ? B / (sigma * sqrtf(w)) : 0.f;
            jj = lane;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float So = __shfl_xor_sync(kFull, S, o);
            const int jo = __shfl_xor_sync(kFull, jj, o);
            if (So > S || (So == S && jo < jj)) { S = So; jj = jo; }
        }
        if (jj != 0x7fffffff) { bs = S; bj = jj; }
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
    if (tid == 0) {
        Partial out;
        out.snr = -CUDART_INF_F; out.k = -1; out.j = -1; out.blk = -1; out.mu = 0.f; out.sigma = 0.f; out.u = -1; out.pad = 0;
        for (int w = 0; w < NW; ++w) {
            if (better(red_s[w], red_i[4 * w], red_i[4 * w + 1], out.snr, out.k, out.j)) {
                out.snr = red_s[w]; out.k = red_i[4 * w]; out.j = red_i[4 * w + 1]; out.u = red_i[4 * w + 2];
                out.mu = red_f[2 * w]; out.sigma = red_f[2 * w + 1];
            }
        }
        P.partials[(size_t)p * slices + sl] = out;
    }
}

size_t search_smem_bytes(int nchan, int RS, int H, int tab_cap)
{
    size_t n = (size_t)nchan * RS + 4 + (size_t)NW * SS + (size_t)NW * H + (size_t)NW * (H >> 5);
    n += (size_t)tab_cap + kWidthBatch + 20 + NW + 4 * NW + 2 * NW + 4;
    return n * sizeof(float) + 16;
}

cudaError_t launch_search(const SearchParams &p, size_t smem_bytes, cudaStream_t st)
{
    const long long blocks = (long long)p.npix * p.n_groups * p.n_wb;
    if (blocks <= 0 || blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    // the opt-in shared-memory size is a per-device function attribute: several plans share it, so only ever raise it
    static size_t granted[64] = {0};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64 && smem_bytes > granted[dev]) {
        e = cudaFuncSetAttribute(k_search, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return e;
        granted[dev] = smem_bytes;
    }
    k_search<<<(unsigned)blocks, NW * 32, smem_bytes, st>>>(p);
    return cudaGetLastError();
}

} // namespace nsfrb
