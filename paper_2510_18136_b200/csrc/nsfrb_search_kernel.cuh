// k_search3: the offline search kernel (steps a1..a6 of DESIGN.md), specialised per plan.
//
// Compiled at the first nsfrb_search of a plan (NVRTC, sm_100a) behind a generated prologue, like k_stream:
//   NCHAN NU NW RS H PITCH NT WMID TRIALS MINB CHAIN16 FUSED   integers (RS raw-tile row stride, H prefix ring length, PITCH workspace row)
//   D_TAB[NU][NCHAN]  delays of the unique trials (dmax ascending)   DMAX_TAB[NU]   K_OF_U[NU]
//   W_TAB[NW]         the usable widths, caller's order (NW <= 32)    J_OF_W[NW]     original width index
//   FUSED             1: the kernel also does the per-pixel reduction and arg-max time (a6), no k_finalize launch
// Same algorithm as the generic k_search (nsfrb_search.cu: one CTA = one pixel x 16 trials, 256-sample blocks,
// cp.async raw prefetch, differential dedispersion, warp = trial, prefix ring in shared memory, exact bound-based
// pruning of wide boxcars), with what the plan fixes folded into the instruction stream:
// One CTA = one pixel x TRIALS trials (a prologue constant: 8 trials = 256 threads lets 2-3 CTAs share an SM).
//   phase 1  every dedispersion operand is rt[immediate]; no change lists in shared memory, no address arithmetic
//   phase 2  the set of widths is static: widths <= 16 from the register window without per-width tests, widths
//            17..WMID from the ring with aligned 128-bit loads (their block bound never prunes: DESIGN.md 5.1),
//            wider ones by branch-and-bound; blocks that lie wholly inside the series skip every validity mask
#ifndef NSFRB_SEARCH_KERNEL_CUH
#define NSFRB_SEARCH_KERNEL_CUH

struct Partial3 { // layout of nsfrb::Partial (nsfrb_internal.h)
    float snr;
    int k, j, blk;
    float mu, sigma;
    int u, pad;
};

struct Search3Params {
    const float *W; // [npix][NCHAN][PITCH] time-contiguous workspace, baseline removed
    Partial3 *partials; // [npix][NGRP]
    int npix;
    // FUSED: the last CTA of a pixel to finish reduces the pixel's partials and finds the arg-max time
    int *counter;   // [npix], zero between launches (the last CTA resets it)
    float *snr_map; // [npix]
    int *argmax;    // [3][npix]
};

namespace s3 {

#define S3_INF __int_as_float(0x7f800000)
constexpr unsigned kFull = 0xffffffffu;
constexpr int NWARP = TRIALS; // trials (= warps) per CTA: 8 or 16
constexpr int LB = 256;    // samples per block
constexpr int SS = 288;    // staging stride per trial: t + 4*(t>>5)
constexpr int NR = H / 32; // ring rows
constexpr int NGRP = (NU + NWARP - 1) / NWARP;

// ring arithmetic: H (and NR = H/32) a power of two turns every wrap into one AND
constexpr bool HP2 = (H & (H - 1)) == 0;
__device__ __forceinline__ int wrapUp(int x) // x in [0, 2H)
{
    if constexpr (HP2) return x & (H - 1);
    else return x >= H ? x - H : x;
}
__device__ __forceinline__ int wrapDn(int x) // x in (-H, H)
{
    if constexpr (HP2) return x & (H - 1);
    else return x < 0 ? x + H : x;
}
__device__ __forceinline__ int wrapR(int r) // r in [0, 2NR)
{
    if constexpr (HP2) return r & (NR - 1);
    else return r >= NR ? r - NR : r;
}

template <int I> struct IC { static constexpr int v = I; };
#define V(x) (decltype(x)::v)
template <int I, int N, class F> __device__ __forceinline__ void sfor(F &&f)
{
    if constexpr (I < N) {
        f(IC<I>{});
        sfor<I + 1, N>(f);
    }
}

// ---- compile-time facts about the width list
__host__ __device__ constexpr int n_small() { int n = 0; for (int j = 0; j < NW; ++j) n += W_TAB[j] <= 16; return n; }
__host__ __device__ constexpr int n_mid() { int n = 0; for (int j = 0; j < NW; ++j) n += (W_TAB[j] > 16 && W_TAB[j] <= WMID); return n; }
__host__ __device__ constexpr int n_large() { int n = 0; for (int j = 0; j < NW; ++j) n += W_TAB[j] > WMID; return n; }
// j-th small / mid width: its index in W_TAB
__host__ __device__ constexpr int small_idx(int q) { int n = 0; for (int j = 0; j < NW; ++j) if (W_TAB[j] <= 16) { if (n == q) return j; ++n; } return 0; }
__host__ __device__ constexpr int mid_idx(int q) { int n = 0; for (int j = 0; j < NW; ++j) if (W_TAB[j] > 16 && W_TAB[j] <= WMID) { if (n == q) return j; ++n; } return 0; }
constexpr int NS = n_small() > 0 ? n_small() : 1;
constexpr int NM = n_mid() > 0 ? n_mid() : 1;

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v)
{
    float r;
    asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
    return r;
}
__device__ __forceinline__ void cp_async16(float *dst, const float *src, int src_bytes)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// raw[c][i] = W[p][c][t0+i] for i < ROWS4 (PITCH is a multiple of 4: aligned 16-byte copies), zero beyond NT.
// Blocks whose rows all lie inside the series take the unchecked path: one pointer pair per channel, static trip count.
template <int ROWS4> __device__ __forceinline__ void issue_raw(const float *Wp, float *raw, int t0, int warp, int lane)
{
    constexpr int ITER = (ROWS4 + 127) / 128;
    if (t0 + ROWS4 <= NT) {
        for (int c = warp; c < NCHAN; c += NWARP) {
            const float *src = Wp + (size_t)c * PITCH + t0 + lane * 4;
            float *dst = raw + c * RS + lane * 4;
#pragma unroll
            for (int k = 0; k < ITER; ++k)
                if (lane * 4 + 128 * k < ROWS4) cp_async16(dst + 128 * k, src + 128 * k, 16);
        }
    } else {
        for (int c = warp; c < NCHAN; c += NWARP) {
            const float *src = Wp + (size_t)c * PITCH;
            float *dst = raw + c * RS;
            for (int i = lane * 4; i < ROWS4; i += 128) {
                const int r = t0 + i;
                int nvalid = NT - r;
                nvalid = nvalid < 0 ? 0 : (nvalid > 4 ? 4 : nvalid);
                cp_async16(dst + i, src + (nvalid ? r : 0), nvalid * 4);
            }
        }
    }
    cp_async_commit();
}

__device__ __forceinline__ bool better(float s, int k, int j, float bs, int bk, int bj)
{
    if (k < 0) return false;
    if (bk < 0) return true;
    if (s != bs) return s > bs;
    if (k != bk) return k < bk;
    return j < bj;
}

// ---- phase 1: differential dedispersion of one block for LEN consecutive trials of group G, starting at trial
// FIRST of the group.  Thread tl (0..255) owns sample tl of the block; rt = raw + tl; so = stage + FIRST*SS + tl + 4*(tl>>5).
// LEN = 8: two chains per 16-trial group run side by side (all 512 threads busy); LEN = 16 (CHAIN16, many channels):
// one chain by half the threads -- the full channel sum of a chain's first trial is paid once instead of twice.
template <int G, int FIRST, int LEN> __device__ __forceinline__ void dedisperse(const float *rt, float *so)
{
    float acc = 0.f;
    sfor<0, LEN>([&](auto s) {
        constexpr int u = G * NWARP + FIRST + V(s);
        if constexpr (u < NU) {
            if constexpr (V(s) == 0) {
                float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
                sfor<0, NCHAN>([&](auto c) {
                    const float v = rt[V(c) * RS + D_TAB[u][V(c)]];
                    if constexpr ((V(c) & 3) == 0) a0 += v;
                    else if constexpr ((V(c) & 3) == 1) a1 += v;
                    else if constexpr ((V(c) & 3) == 2) a2 += v;
                    else a3 += v;
                });
                acc = (a0 + a1) + (a2 + a3);
            } else {
                float a0 = 0.f, a1 = 0.f;
                sfor<0, NCHAN>([&](auto c) {
                    if constexpr (D_TAB[u][V(c)] != D_TAB[u - 1][V(c)]) {
                        const float v = rt[V(c) * RS + D_TAB[u][V(c)]] - rt[V(c) * RS + D_TAB[u - 1][V(c)]];
                        if constexpr ((V(c) & 1) == 0) a0 += v; else a1 += v;
                    }
                });
                acc += a0 + a1;
            }
            so[V(s) * SS] = acc;
        }
    });
}

// ---- phase 2 state of one warp (= one trial)
struct Trial {
    float M;      // lane j: running max_t of width j for the large widths (and the final per-width max for all)
    float ms[NS]; // per-lane running maxima of the small widths (<= 16), reduced over lanes at the end
    float mm[NM]; // the same for the mid widths (17..WMID)
    float mu0, s1, s2, carry;
    int tpos, rr;
};

template <bool INSIDE>
__device__ __forceinline__ void search_block(Trial &T, const float *stage_row, float *ring, float *rmin, int lane, int t0, int T_k,
                                             int wl, bool is_large)
{
    // INSIDE: the whole block lies inside the series (t0 + LB <= T_k): no validity masks anywhere
    float p8[8];
    {
        const float4 *sp = reinterpret_cast<const float4 *>(stage_row + 8 * lane + 4 * (lane >> 2));
        const float4 xa = sp[0], xb = sp[1];
        p8[0] = xa.x; p8[1] = xa.y; p8[2] = xa.z; p8[3] = xa.w;
        p8[4] = xb.x; p8[5] = xb.y; p8[6] = xb.z; p8[7] = xb.w;
    }
    const int tb = t0 + 8 * lane;
    const int nv = T_k - tb; // sample i of this lane is valid iff i < nv
    if (t0 == 0) {
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) s += (INSIDE || i < nv) ? p8[i] : 0.f;
        T.mu0 = warp_sum(s) / (float)(T_k < LB ? T_k : LB);
    }
    float run = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float x = (INSIDE || i < nv) ? p8[i] - T.mu0 : 0.f;
        T.s1 += x;
        T.s2 = fmaf(x, x, T.s2);
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
    const float base = T.carry + excl;
#pragma unroll
    for (int i = 0; i < 8; ++i) p8[i] += base; // P[t+1], t = tb + i
    T.carry = __shfl_sync(kFull, p8[7], 31);

    int sb = T.tpos + 8 * lane; // ring slot of sample tb (8 | H: the 8 slots never straddle the wrap)
    sb = wrapUp(sb);
    {
        float4 *rp = reinterpret_cast<float4 *>(ring + sb);
        rp[0] = make_float4(p8[0], p8[1], p8[2], p8[3]);
        rp[1] = make_float4(p8[4], p8[5], p8[6], p8[7]);
        if constexpr (n_large() > 0) {
            float lmin = fminf(fminf(fminf(p8[0], p8[1]), fminf(p8[2], p8[3])), fminf(fminf(p8[4], p8[5]), fminf(p8[6], p8[7])));
            lmin = fminf(lmin, __shfl_xor_sync(kFull, lmin, 1));
            lmin = fminf(lmin, __shfl_xor_sync(kFull, lmin, 2));
            if ((lane & 3) == 0) rmin[sb >> 5] = lmin;
        }
    }
    __syncwarp();

    // ends of this lane: E[i] = P[tb+i+1], -inf where the end lies beyond the series
    float E[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) E[i] = (INSIDE || i < nv) ? p8[i] : -S3_INF;

    // ---- widths <= 16 from a 24-sample register window
    if constexpr (n_small() > 0) {
        float Wn[24];
#pragma unroll
        for (int i = 0; i < 8; ++i) Wn[16 + i] = p8[i];
        int s2b = sb - 16, s1b = sb - 8;
        s2b = wrapDn(s2b);
        s1b = wrapDn(s1b);
        const float4 *w2 = reinterpret_cast<const float4 *>(ring + s2b);
        const float4 *w1 = reinterpret_cast<const float4 *>(ring + s1b);
        const float4 a = w2[0], b = w2[1], c = w1[0], d = w1[1];
        Wn[0] = a.x; Wn[1] = a.y; Wn[2] = a.z; Wn[3] = a.w; Wn[4] = b.x; Wn[5] = b.y; Wn[6] = b.z; Wn[7] = b.w;
        Wn[8] = c.x; Wn[9] = c.y; Wn[10] = c.z; Wn[11] = c.w; Wn[12] = d.x; Wn[13] = d.y; Wn[14] = d.z; Wn[15] = d.w;
        sfor<0, n_small()>([&](auto q) {
            constexpr int w = W_TAB[small_idx(V(q))];
            float m = T.ms[V(q)];
#pragma unroll
            for (int i = 0; i < 8; ++i) m = fmaxf(m, E[i] - Wn[16 + i - w]);
            T.ms[V(q)] = m;
        });
    }
    // ---- widths 17..WMID straight from the ring: starts of this lane's 8 ends are 8 consecutive slots from
    //      sb - w; read the 3 aligned float4 that cover them (the misalignment (-w) & 3 is static)
    if constexpr (n_mid() > 0) {
        sfor<0, n_mid()>([&](auto q) {
            constexpr int w = W_TAB[mid_idx(V(q))];
            constexpr int r = (4 - (w & 3)) & 3; // (sb - w) mod 4, sb being a multiple of 8
            int a0 = sb - w - r;                 // aligned slot of the first float4
            a0 = wrapDn(a0);
            int a1 = a0 + 4, a2 = a0 + 8;
            a1 = wrapUp(a1);
            a2 = wrapUp(a2);
            const float4 x0 = *reinterpret_cast<const float4 *>(ring + a0);
            const float4 x1 = *reinterpret_cast<const float4 *>(ring + a1);
            float v[12] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w, 0.f, 0.f, 0.f, 0.f};
            if constexpr (r != 0) {
                const float4 x2 = *reinterpret_cast<const float4 *>(ring + a2);
                v[8] = x2.x; v[9] = x2.y; v[10] = x2.z; v[11] = x2.w;
            }
            float m = T.mm[V(q)];
#pragma unroll
            for (int i = 0; i < 8; ++i) m = fmaxf(m, E[i] - v[r + i]);
            T.mm[V(q)] = m;
        });
    }
    // ---- widths > WMID: bound, then evaluate only the blocks that can raise the maximum
    if constexpr (n_large() > 0) {
        float Pe[8], emx = -S3_INF;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            int pos = T.tpos + lane + 32 * i;
            pos = wrapUp(pos);
            const float v = (INSIDE || t0 + lane + 32 * i + 1 <= T_k) ? ring[pos] : -S3_INF;
            Pe[i] = v;
            emx = fmaxf(emx, v);
        }
        const float Emax = warp_max(emx);
        bool surv = false;
        if (is_large) {
            float mn = S3_INF;
            int r = T.rr;
#pragma unroll
            for (int q = 0; q < 9; ++q) {
                mn = fminf(mn, rmin[r]);
                r = wrapR(r + 1);
            }
            surv = (Emax - mn) > T.M;
        }
        unsigned mask = __ballot_sync(kFull, surv);
        while (mask) {
            const int j = __ffs(mask) - 1;
            mask &= mask - 1;
            int q = T.tpos - W_TAB[j]; // ring slot of the start that belongs to end slot tpos
            q = wrapDn(q);
            float v = -S3_INF;
            if (q + LB <= H) {
                const float *b = ring + q + lane;
#pragma unroll
                for (int i = 0; i < 8; ++i) v = fmaxf(v, Pe[i] - b[32 * i]);
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    int a = q + lane + 32 * i;
                    a = wrapUp(a);
                    v = fmaxf(v, Pe[i] - ring[a]);
                }
            }
            v = warp_max(v);
            if (lane == j) T.M = fmaxf(T.M, v);
        }
    }
    __syncwarp();
}

// ---- a6, last step, fused: best group of the pixel, then the arg-max time by recomputing the winning series
// (L2-hot: the pixel's CTAs have just read it) over the starts that can hold it, with the mean/sigma the search found.
__device__ __forceinline__ void finalize_pixel(const Search3Params &P, float *fs, int p)
{
    constexpr int NTHR = NWARP * 32, PER = NTHR / 32;
    float *sc_f = fs + NT + 2;                        // [NTHR]
    int *sc_i = reinterpret_cast<int *>(sc_f + NTHR); // [NTHR]
    __shared__ Partial3 best;
    const int tid = threadIdx.x;
    if (tid == 0) {
        Partial3 b;
        b.snr = -S3_INF; b.k = -1; b.j = -1; b.blk = -1; b.mu = 0.f; b.sigma = 0.f; b.u = -1; b.pad = 0;
        const int4 *pp = reinterpret_cast<const int4 *>(P.partials + (size_t)p * NGRP);
        for (int g = 0; g < NGRP; ++g) {
            const int4 lo = __ldcg(pp + 2 * g), hi = __ldcg(pp + 2 * g + 1); // written by other CTAs: bypass L1
            const float snr = __int_as_float(lo.x);
            if (better(snr, lo.y, lo.z, b.snr, b.k, b.j)) {
                b.snr = snr; b.k = lo.y; b.j = lo.z; b.blk = lo.w;
                b.mu = __int_as_float(hi.x); b.sigma = __int_as_float(hi.y); b.u = hi.z; b.pad = hi.w;
            }
        }
        best = b;
    }
    __syncthreads();
    const Partial3 b = best;
    if (b.k < 0) {
        if (tid == 0) {
            P.snr_map[p] = -S3_INF;
            P.argmax[p] = -1; P.argmax[(size_t)P.npix + p] = -1; P.argmax[2 * (size_t)P.npix + p] = -1;
        }
        return;
    }
    const int w = W_TAB[b.j];
    const int T = NT - DMAX_TAB[b.u];
    const int n = T; // samples [0, T): every start 0..T-w is a candidate
    const float *Wp = P.W + (size_t)p * NCHAN * (size_t)PITCH;
    for (int i = tid; i < n; i += NTHR) {
        float s0 = 0.f, s1 = 0.f;
        sfor<0, NCHAN>([&](auto c) {
            const float v = __ldg(Wp + (size_t)V(c) * PITCH + i + D_TAB[b.u][V(c)]);
            if constexpr ((V(c) & 1) == 0) s0 += v; else s1 += v;
        });
        fs[i + 1] = (s0 + s1) - b.mu;
    }
    if (tid == 0) fs[0] = 0.f;
    __syncthreads();
    // block-wide inclusive scan of fs[1..n]: odd-length chunk per thread (conflict-free)
    const int ch = ((n + NTHR - 1) / NTHR) | 1;
    const int a0 = 1 + tid * ch, a1 = (a0 + ch < n + 1) ? a0 + ch : n + 1;
    float tot = 0.f;
    for (int i = a0; i < a1; ++i) tot += fs[i];
    sc_f[tid] = tot;
    __syncthreads();
    if (tid < 32) { // scan of the NTHR chunk totals by one warp, PER per lane
        float v[PER], run = 0.f;
#pragma unroll
        for (int i = 0; i < PER; ++i) { v[i] = sc_f[tid * PER + i]; run += v[i]; }
        float incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const float y = __shfl_up_sync(kFull, incl, o);
            if (tid >= o) incl += y;
        }
        float ex = incl - run;
#pragma unroll
        for (int i = 0; i < PER; ++i) { sc_f[tid * PER + i] = ex; ex += v[i]; }
    }
    __syncthreads();
    {
        float run = sc_f[tid];
        for (int i = a0; i < a1; ++i) { run += fs[i]; fs[i] = run; }
    }
    __syncthreads();
    // arg-max over starts i in [0, n-w]: B = P[i+w] - P[i], smallest i on ties
    float bv = -S3_INF;
    int bi = 0x7fffffff;
    for (int i = tid; i <= n - w; i += NTHR) {
        const float B = fs[i + w] - fs[i];
        if (B > bv) { bv = B; bi = i; }
    }
    sc_f[tid] = bv; sc_i[tid] = bi;
    __syncthreads();
    for (int o = NTHR / 2; o > 0; o >>= 1) {
        if (tid < o) {
            const float ov = sc_f[tid + o]; const int oi = sc_i[tid + o];
            if (ov > sc_f[tid] || (ov == sc_f[tid] && oi < sc_i[tid])) { sc_f[tid] = ov; sc_i[tid] = oi; }
        }
        __syncthreads();
    }
    if (tid == 0) {
        const float B = sc_f[0];
        const float S = b.sigma > 0.f ? B / (b.sigma * sqrtf((float)w)) : 0.f;
        P.snr_map[p] = S;
        P.argmax[p] = b.k;
        P.argmax[(size_t)P.npix + p] = J_OF_W[b.j];
        P.argmax[2 * (size_t)P.npix + p] = sc_i[0];
    }
}

constexpr int kSmemFloats = NCHAN * RS + 4 + NWARP * SS + NWARP * H + NWARP * NR + NWARP * 8;

template <int G> __device__ __forceinline__ void run_group(const Search3Params &P, float *smem, int p)
{
    float *raw = smem;                      // [NCHAN][RS] (+4 pad)
    float *stage = raw + NCHAN * RS + 4;    // [NWARP][SS]  padded: index t + 4*(t>>5)
    float *rings = stage + NWARP * SS;      // [NWARP][H]   P[t+1] at slot t mod H
    float *rmins = rings + NWARP * H;       // [NWARP][NR]  min of P over each 32-slot row
    float *red = rmins + NWARP * NR;        // [NWARP][8]   per-trial results

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int u = G * NWARP + warp;
    const bool has = u < NU && (NT - DMAX_TAB[u < NU ? u : NU - 1]) >= 1;
    const int T_k = has ? NT - DMAX_TAB[u] : 0;
    float *ring = rings + warp * H;
    float *rmin = rmins + warp * NR;

    // group facts (static): the largest delay and the longest series
    constexpr int ulast = (G * NWARP + NWARP - 1 < NU) ? G * NWARP + NWARP - 1 : NU - 1;
    constexpr int dmax_g = DMAX_TAB[ulast];     // trials are sorted by dmax
    constexpr int T_g = NT - DMAX_TAB[G * NWARP]; // longest series of the group
    constexpr int rows4 = (LB + dmax_g + 3) & ~3;

    // "before time 0": only the slots a start can reach from the first blocks need the +inf marker -- the last
    // INIT slots of the ring (widest width + the 32-slot rows the bound looks at); the rest is written before it is read
    constexpr int WMAXS = []() { int m = 1; for (int j = 0; j < NW; ++j) m = (W_TAB[j] > m && W_TAB[j] < H) ? W_TAB[j] : m; return m; }();
    constexpr int INIT = ((WMAXS + 95) / 32) * 32 < H ? ((WMAXS + 95) / 32) * 32 : H;
    for (int i = H - INIT + lane; i < H; i += 32) ring[i] = (i == H - 1) ? 0.f : S3_INF; // P[0] = 0 at slot -1
    for (int i = NR - INIT / 32 + lane; i < NR; i += 32) rmin[i] = (i == NR - 1) ? 0.f : S3_INF;

    const int wl = lane < NW ? W_TAB[lane] : 0;
    const bool is_large = wl > WMID;
    Trial T;
    T.M = -S3_INF;
#pragma unroll
    for (int q = 0; q < NS; ++q) T.ms[q] = -S3_INF;
#pragma unroll
    for (int q = 0; q < NM; ++q) T.mm[q] = -S3_INF;
    T.mu0 = 0.f; T.s1 = 0.f; T.s2 = 0.f; T.carry = 0.f; T.tpos = 0;
    T.rr = ((-wl) >> 5) + NR; // ring row of the first start of block 0 (floor division)
    if (T.rr >= NR || T.rr < 0) T.rr = 0;

    const float *Wp = P.W + (size_t)p * NCHAN * (size_t)PITCH;
    if (T_g > 0) issue_raw<rows4>(Wp, raw, 0, warp, lane);
    __syncthreads();

    for (int t0 = 0; t0 < T_g; t0 += LB) {
        cp_async_wait_all();
        __syncthreads(); // raw(b) landed; every warp is done with stage(b-1)
        {
            const int tl = tid & (LB - 1);
            const float *rt = raw + tl;
            float *so = stage + tl + 4 * (tl >> 5);
            if constexpr (NWARP == 8) {
                dedisperse<G, 0, 8>(rt, so);
            } else if constexpr (CHAIN16) {
                if (tid < LB) dedisperse<G, 0, 16>(rt, so);
            } else {
                if (tid < LB) dedisperse<G, 0, 8>(rt, so);
                else dedisperse<G, 8, 8>(rt, so + 8 * SS);
            }
        }
        __syncthreads(); // stage(b) complete; the raw tile is free again
        if (t0 + LB < T_g) issue_raw<rows4>(Wp, raw, t0 + LB, warp, lane);

        if (has && t0 < T_k) {
            if (t0 + LB <= T_k) search_block<true>(T, stage + warp * SS, ring, rmin, lane, t0, T_k, wl, is_large);
            else search_block<false>(T, stage + warp * SS, ring, rmin, lane, t0, T_k, wl, is_large);
        }
        T.tpos += LB;
        T.tpos = wrapUp(T.tpos);
        T.rr += LB / 32;
        T.rr = wrapR(T.rr);
    }

    // ---- a6 (per trial): exact mean / variance, normalise, best width
    float bs = -S3_INF;
    int bj = -1;
    float mu = 0.f, sigma = 0.f;
    if (has) {
        const float S1 = warp_sum(T.s1), S2 = warp_sum(T.s2);
        const float invT = 1.f / (float)T_k;
        const float delta = S1 * invT;
        const float var = fmaxf(fmaf(-delta, delta, S2 * invT), 0.f);
        sigma = sqrtf(var);
        mu = T.mu0 + delta;
        float M = T.M;
        sfor<0, n_small()>([&](auto q) {
            const float v = warp_max(T.ms[V(q)]);
            if (lane == small_idx(V(q))) M = v;
        });
        sfor<0, n_mid()>([&](auto q) {
            const float v = warp_max(T.mm[V(q)]);
            if (lane == mid_idx(V(q))) M = v;
        });
        float S = -S3_INF;
        int jj = 0x7fffffff;
        if (lane < NW && M > -S3_INF) {
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
        red[warp * 8 + 0] = bs;
        reinterpret_cast<int *>(red)[warp * 8 + 1] = (has && bj >= 0) ? K_OF_U[u] : -1;
        reinterpret_cast<int *>(red)[warp * 8 + 2] = bj;
        reinterpret_cast<int *>(red)[warp * 8 + 3] = u;
        red[warp * 8 + 4] = mu;
        red[warp * 8 + 5] = sigma;
    }
    __syncthreads();
    if (tid == 0) {
        Partial3 out;
        out.snr = -S3_INF; out.k = -1; out.j = -1; out.blk = -1; out.mu = 0.f; out.sigma = 0.f; out.u = -1; out.pad = 0;
        for (int w = 0; w < NWARP; ++w) {
            const float s = red[w * 8 + 0];
            const int k = reinterpret_cast<int *>(red)[w * 8 + 1], j = reinterpret_cast<int *>(red)[w * 8 + 2];
            if (better(s, k, j, out.snr, out.k, out.j)) {
                out.snr = s; out.k = k; out.j = j; out.u = reinterpret_cast<int *>(red)[w * 8 + 3];
                out.mu = red[w * 8 + 4]; out.sigma = red[w * 8 + 5];
            }
        }
        P.partials[(size_t)p * NGRP + G] = out;
    }
#if FUSED
    __shared__ int is_last;
    if (tid == 0) {
        __threadfence(); // the partial is visible before the ticket is taken
        const int prev = atomicAdd(P.counter + p, 1);
        is_last = (prev == NGRP - 1);
        if (is_last) P.counter[p] = 0; // ready for the next launch
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        finalize_pixel(P, smem, p);
    }
#endif
}

template <int G0, int N> __device__ __forceinline__ void dispatch(int g, const Search3Params &P, float *smem, int p)
{
    if constexpr (N == 1) {
        run_group<G0>(P, smem, p);
    } else {
        if (g < G0 + N / 2) dispatch<G0, N / 2>(g, P, smem, p);
        else dispatch<G0 + N / 2, N - N / 2>(g, P, smem, p);
    }
}

} // namespace s3

extern "C" __global__ void __launch_bounds__(s3::NWARP * 32, MINB) k_search3(const Search3Params P)
{
    extern __shared__ __align__(16) float smem[];
    const int p = blockIdx.x / s3::NGRP;
    const int g = blockIdx.x - p * s3::NGRP;
    s3::dispatch<0, s3::NGRP>(g, P, smem, p);
}

#endif
