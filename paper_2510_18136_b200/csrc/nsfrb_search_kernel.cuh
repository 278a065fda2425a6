// k_search4: the offline search kernel (steps a1..a6 of DESIGN.md), specialised per plan.
//
// Compiled at nsfrb_plan_prepare / the first nsfrb_search of a plan (NVRTC, sm_100a) behind a generated prologue:
//   NCHAN NU NW NWARP PXI H PITCH DPITCH NT WMID SDIR PRUNE   integers
//                     NWARP trials (= warps) per CTA, PXI pixels per work item, H prefix ring length (a multiple of 64), PITCH
//                     workspace row, DPITCH row of the dedispersed scratch, WMID/SDIR width classes (below), PRUNE = 0 switches
//                     the bounds off (every cell is evaluated)
//   D_TAB[NU][NCHAN]  delays of the unique trials (dmax ascending)   DMAX_TAB[NU]   K_OF_U[NU]
//   W_TAB[NW]         the usable widths, caller's order (NW <= 32)    J_OF_W[NW]     original width index
//
// Persistent CTAs; a work item = PXI pixels x NWARP trials, in three phases with one CTA barrier between them:
//   sweep A (thread = 4 consecutive samples)  differential dedispersion along the DM axis straight from the time-contiguous batch
//            workspace: per channel one aligned window of vector loads (immediate offsets) covers every delay of the group; the
//            first trial is the plain channel sum, every next one adds (new - previous trial's) for the channels whose delay
//            changed.  D goes to a per-CTA scratch (L2-resident) as float4.
//   sweep B (warp = trial, pixel after pixel; no barrier)  first one pass over the series for its exact mean and sigma
//            (a1, a3), then blocks of 256 samples, 8 consecutive samples per lane: x = D - mu, prefix by 8 serial adds + one
//            warp scan, P into the trial's ring (two interleaved planes of float4: every 128-bit access of a warp is
//            conflict-free), 8-sample minima beside it.  Because sigma is known, every boxcar is worth a known S/N, and a
//            cell matters only if it can reach the best S/N found so far for the pixel (S*, shared by the CTA's warps):
//              widths <= SDIR        every cell, from the register window
//              widths SDIR+1..16     bound: max of the lane's 8 ends - min of the 16 samples before them and its own 8
//              widths 17..WMID       bound: max of the 8 ends - min of the two 8-sample groups holding the starts
//              widths > WMID         lane j bounds width j for the whole block from 32-sample row minima
//            All bounds of a block are formed side by side (independent loads, no branches) into one bit mask, OR-reduced
//            over the warp; only the widths whose bit is set read the ring and evaluate their cells.  Every skipped cell is
//            below its bound, hence below S* <= the final maximum: the maximum and its (k, j, t) are exact.
//            End of a series: S = (M - w delta)/(sigma sqrt(w)) per width, best width of the trial (a6).
//   tail     warp q takes pixel q: best trial of the group, then the arg-max time by running the prefix of the winning
//            series once more (same operations, so the same P bit for bit) into its scratch row and scanning the one
//            width; the partial (S, k, j, t) goes to global memory, and the last CTA of a pixel (ticket) writes the pixel's
//            outputs.
#ifndef NSFRB_SEARCH_KERNEL_CUH
#define NSFRB_SEARCH_KERNEL_CUH

struct Partial4 { // layout of nsfrb::Partial (nsfrb_internal.h)
    float snr;
    int k, j, t; // t: window start of the maximum
    float mu, sigma;
    int u, pad;
};

struct Search4Params {
    const float *W;     // [npb][NCHAN][PITCH] time-contiguous workspace of this batch, baseline removed
    Partial4 *partials; // [npix][NGRP]
    int npix;           // pixels of the image (stride of the outputs)
    int p0, npb;        // this launch searches pixels [p0, p0 + npb)
    int *counter;       // [npix] tickets, zero between launches (the last CTA of a pixel resets its own)
    float *snr_map;     // [npix]
    int *argmax;        // [3][npix]
    float *scratch;     // [gridDim.x][PXI][NWARP][DPITCH] dedispersed series of the item in flight
};

namespace s4 {

#define S4_INF __int_as_float(0x7f800000)
constexpr unsigned kFull = 0xffffffffu;
constexpr int NTHR = NWARP * 32;
constexpr int LB = 256;    // samples per block of sweep B
constexpr int NR = H / 32; // ring rows of 32 slots
constexpr int NG = H / 8;  // ring groups of 8 slots (one lane's samples of a block)
constexpr int NGRP = (NU + NWARP - 1) / NWARP;
constexpr int PL1 = H / 2 + 16; // the ring's second plane: float4 chunk q of the series sits at (q & 1)*PL1 + 4*(q >> 1)
constexpr int RINGF = H + 16;

constexpr bool HP2 = (H & (H - 1)) == 0;
__device__ __forceinline__ int wrapG(int g) // g in (-NG, 2NG)
{
    if constexpr (HP2) return g & (NG - 1);
    else return g < 0 ? g + NG : (g >= NG ? g - NG : g);
}
__device__ __forceinline__ int wrapR(int r) // r in [0, 2NR)
{
    if constexpr (HP2) return r & (NR - 1);
    else return r >= NR ? r - NR : r;
}
// physical float index of logical ring slot s in [0, H)
__device__ __forceinline__ int slot_addr(int s) { return ((s >> 2) & 1) * PL1 + 4 * (s >> 3) + (s & 3); }

template <int I> struct IC { static constexpr int v = I; };
#define V(x) (decltype(x)::v)
template <int I, int N, class F> __device__ __forceinline__ void sfor(F &&f)
{
    if constexpr (I < N) {
        f(IC<I>{});
        sfor<I + 1, N>(f);
    }
}

// ---- compile-time facts about the width list: class 0 direct (<= SDIR), 1 window (SDIR+1..16), 2 mid (17..WMID), 3 large
__host__ __device__ constexpr int wclass(int w) { return w <= SDIR ? 0 : (w <= 16 ? 1 : (w <= WMID ? 2 : 3)); }
__host__ __device__ constexpr int n_class(int c) { int n = 0; for (int j = 0; j < NW; ++j) n += wclass(W_TAB[j]) == c; return n; }
__host__ __device__ constexpr int class_idx(int c, int q) { int n = 0; for (int j = 0; j < NW; ++j) if (wclass(W_TAB[j]) == c) { if (n == q) return j; ++n; } return 0; }
__host__ __device__ constexpr unsigned class_mask(int c) { unsigned m = 0; for (int j = 0; j < NW; ++j) if (wclass(W_TAB[j]) == c) m |= 1u << j; return m; }
constexpr int ND = n_class(0), NWN = n_class(1), NM = n_class(2), NL = n_class(3);
__host__ __device__ constexpr float csqrt(int w) // sqrt(w) (Newton in double, rounded to float)
{
    double x = (double)w, r = x > 1.0 ? x / 2 : 1.0;
    for (int i = 0; i < 40; ++i) r = 0.5 * (r + x / r);
    return (float)r;
}

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
__device__ __forceinline__ bool better(float s, int k, int j, float bs, int bk, int bj)
{
    if (k < 0) return false;
    if (bk < 0) return true;
    if (s != bs) return s > bs;
    if (k != bk) return k < bk;
    return j < bj;
}

// ---- sweep A: differential dedispersion of SPT consecutive samples t .. t + SPT - 1 (t a multiple of SPT) for the NWARP trials
// of group G.  wp = W[p] + t; dst = scratch + t.  Channel by channel the thread loads ONE aligned window that covers every
// delay of the group (2-4 vector loads instead of one scalar load per (trial, changed channel)) and adds, for each trial,
// window[new delay] - window[previous trial's delay] to that trial's difference; the first trial takes the plain sum.  The
// dedispersed values are the running sum of the differences over the trials.
constexpr int SPT = NWARP <= 16 ? 4 : 2; // samples per thread (the differences of all trials live in registers)

template <int G, int C> struct ChanSpan { // delays of channel C over the trials of group G
    static __host__ __device__ constexpr int lo() { int m = 1 << 30; for (int s = 0; s < NWARP; ++s) { const int u = G * NWARP + s; if (u < NU && D_TAB[u][C] < m) m = D_TAB[u][C]; } return m; }
    static __host__ __device__ constexpr int hi() { int m = 0; for (int s = 0; s < NWARP; ++s) { const int u = G * NWARP + s; if (u < NU && D_TAB[u][C] > m) m = D_TAB[u][C]; } return m; }
};

template <int G> __device__ __forceinline__ void dedisperse(const float *__restrict__ wp, float *__restrict__ dst)
{
    float diff[NWARP][SPT];
#pragma unroll
    for (int s = 0; s < NWARP; ++s)
#pragma unroll
        for (int i = 0; i < SPT; ++i) diff[s][i] = 0.f;
    sfor<0, NCHAN>([&](auto c) {
        constexpr int a = ChanSpan<G, V(c)>::lo() / SPT * SPT;                 // aligned start of the window
        constexpr int nq = (ChanSpan<G, V(c)>::hi() + SPT - 1 - a) / SPT + 1;   // vectors that cover [lo, hi + SPT - 1]
        float win[nq * SPT];
        sfor<0, nq>([&](auto q) {
            if constexpr (SPT == 4) {
                const float4 v = __ldg(reinterpret_cast<const float4 *>(wp + V(c) * PITCH + a) + V(q));
                win[4 * V(q)] = v.x; win[4 * V(q) + 1] = v.y; win[4 * V(q) + 2] = v.z; win[4 * V(q) + 3] = v.w;
            } else {
                const float2 v = __ldg(reinterpret_cast<const float2 *>(wp + V(c) * PITCH + a) + V(q));
                win[2 * V(q)] = v.x; win[2 * V(q) + 1] = v.y;
            }
        });
        sfor<0, NWARP>([&](auto s) {
            constexpr int u = G * NWARP + V(s);
            if constexpr (u < NU) {
                if constexpr (V(s) == 0) {
#pragma unroll
                    for (int i = 0; i < SPT; ++i) diff[0][i] += win[D_TAB[u][V(c)] - a + i];
                } else if constexpr (D_TAB[u][V(c)] != D_TAB[u - 1][V(c)]) {
#pragma unroll
                    for (int i = 0; i < SPT; ++i) diff[V(s)][i] += win[D_TAB[u][V(c)] - a + i] - win[D_TAB[u - 1][V(c)] - a + i];
                }
            }
        });
    });
    float acc[SPT];
#pragma unroll
    for (int i = 0; i < SPT; ++i) acc[i] = 0.f;
    sfor<0, NWARP>([&](auto s) {
        if constexpr (G * NWARP + V(s) < NU) {
#pragma unroll
            for (int i = 0; i < SPT; ++i) acc[i] += diff[V(s)][i];
            if constexpr (SPT == 4) *reinterpret_cast<float4 *>(dst + V(s) * DPITCH) = make_float4(acc[0], acc[1], acc[2], acc[3]);
            else *reinterpret_cast<float2 *>(dst + V(s) * DPITCH) = make_float2(acc[0], acc[1]);
        }
    });
}

// ---- sweep B state of one warp (= one trial)
struct Trial {
    float md[ND > 0 ? ND : 1];   // per-lane running maxima of the direct widths
    float mw[NWN > 0 ? NWN : 1]; // ... of the window widths
    float mm[NM > 0 ? NM : 1];   // ... of the mid widths
    float ML;                    // lane j: running maximum of large width j (warp-wide)
    float mu, sigma, rsig, carry;
    float sbest, thr;            // the CTA's best S/N as this warp last saw it; the prefix-unit threshold per sqrt(w)
    int g0, rr;                  // ring group of lane 0 in this block; NR - ceil(w/32) of the lane's large width
};

// three (two) aligned float4 of the ring that hold the starts of the lane's 8 ends for width w > 8; max over the 8 cells
template <int w> __device__ __forceinline__ float eval_far(const float *ring, int g, const float (&E)[8])
{
    constexpr int a = (4 - (w & 3)) & 3; // first start slot = 8g - w = 4*q0 + a
    constexpr int c = (w + a) / 4;       // q0 = 2g - c
    float v[12] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    sfor<0, (a ? 3 : 2)>([&](auto i) {
        constexpr int plane = (((c + V(i)) % 2) + 2) % 2; // chunk q0 + i = 2g - c + i
        constexpr int off = (V(i) - c - plane) / 2;       // its group relative to g (exact, <= 0)
        const int pos = wrapG(g + off);
        const float4 x = *reinterpret_cast<const float4 *>(ring + plane * PL1 + 4 * pos);
        v[4 * V(i)] = x.x; v[4 * V(i) + 1] = x.y; v[4 * V(i) + 2] = x.z; v[4 * V(i) + 3] = x.w;
    });
    float m = -S4_INF;
#pragma unroll
    for (int i = 0; i < 8; ++i) m = fmaxf(m, E[i] - v[a + i]);
    return m;
}

// the CTA's best S/N: monotone, shared through one word of shared memory (S >= 0: integer order = float order)
__device__ __forceinline__ void publish(Trial &T, int *sbest, float S, int lane)
{
    if (S > T.sbest) {
        T.sbest = S;
        if (lane == 0) atomicMax(sbest, __float_as_int(S));
    }
}

template <bool INSIDE>
__device__ __forceinline__ void search_block(Trial &T, float (&p8)[8], float *ring, float *rm8, float *rm32, int *sbest, int lane, int t0,
                                             int T_k, float sqw_lane, bool is_large)
{
    // INSIDE: the whole block lies inside the series (t0 + LB <= T_k): no validity masks anywhere
    const int tb = t0 + 8 * lane;
    const int nv = T_k - tb; // sample i of this lane is valid iff i < nv
    float run = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float x = (INSIDE || i < nv) ? p8[i] - T.mu : 0.f;
        run += x;
        p8[i] = run;
    }
    // exclusive scan of the lane totals in three rounds of independent shuffles (sums of 4, of 16, of 32 lanes)
    float ex;
    {
        float a = __shfl_up_sync(kFull, run, 1);
        if (lane == 0) a = 0.f;
        const float y1 = __shfl_up_sync(kFull, a, 1), y2 = __shfl_up_sync(kFull, a, 2), y3 = __shfl_up_sync(kFull, a, 3);
        const float s4 = (a + (lane >= 1 ? y1 : 0.f)) + ((lane >= 2 ? y2 : 0.f) + (lane >= 3 ? y3 : 0.f));
        const float z1 = __shfl_up_sync(kFull, s4, 4), z2 = __shfl_up_sync(kFull, s4, 8), z3 = __shfl_up_sync(kFull, s4, 12);
        const float s16 = (s4 + (lane >= 4 ? z1 : 0.f)) + ((lane >= 8 ? z2 : 0.f) + (lane >= 12 ? z3 : 0.f));
        const float q = __shfl_up_sync(kFull, s16, 16);
        ex = s16 + (lane >= 16 ? q : 0.f);
    }
    const float base = T.carry + ex;
#pragma unroll
    for (int i = 0; i < 8; ++i) p8[i] += base; // P[t+1], t = tb + i
    T.carry = __shfl_sync(kFull, p8[7], 31);

    const int g = wrapG(T.g0 + lane); // ring group of this lane's 8 samples
    // ends of this lane: E[i] = P[tb+i+1], -inf where the end lies beyond the series
    float E[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) E[i] = (INSIDE || i < nv) ? p8[i] : -S4_INF;
    const float M8 = fmaxf(fmaxf(fmaxf(E[0], E[1]), fmaxf(E[2], E[3])), fmaxf(fmaxf(E[4], E[5]), fmaxf(E[6], E[7])));
    const float m8own = fminf(fminf(fminf(p8[0], p8[1]), fminf(p8[2], p8[3])), fminf(fminf(p8[4], p8[5]), fminf(p8[6], p8[7])));
    {
        *reinterpret_cast<float4 *>(ring + 4 * g) = make_float4(p8[0], p8[1], p8[2], p8[3]);
        *reinterpret_cast<float4 *>(ring + PL1 + 4 * g) = make_float4(p8[4], p8[5], p8[6], p8[7]);
        rm8[g] = m8own;      // minima of the 8-slot groups, kept twice so that "g + NG - offset" never wraps
        rm8[g + NG] = m8own;
        if constexpr (NL > 0) {
            float lmin = fminf(m8own, __shfl_xor_sync(kFull, m8own, 1));
            lmin = fminf(lmin, __shfl_xor_sync(kFull, lmin, 2));
            if ((lane & 3) == 0) { rm32[g >> 2] = lmin; rm32[(g >> 2) + NR] = lmin; } // twice, like the 8-slot minima
        }
    }
    __syncwarp();

    const float *rmg = rm8 + g + NG;
    const float thr = T.thr; // B >= thr*sqrt(w)  <=>  the cell can reach S* (as of the previous block; a hair below, for rounding)

    // ---- the bounds of every width that is not evaluated unconditionally, side by side, into one bit per width
    unsigned bits = 0;
    if constexpr (PRUNE) {
        if constexpr (NWN > 0) { // starts of the window widths: the 16 samples before the lane's first end, and its own 8
            const float bnd = M8 - fminf(fminf(rmg[-2], rmg[-1]), m8own);
            sfor<0, NWN>([&](auto q) {
                constexpr int j = class_idx(1, V(q));
                if (bnd >= thr * csqrt(W_TAB[j])) bits |= 1u << j;
            });
        }
        if constexpr (NM > 0) { // starts of the lane's 8 ends lie in the two 8-slot groups from 8g - w
            sfor<0, NM>([&](auto q) {
                constexpr int j = class_idx(2, V(q));
                constexpr int w = W_TAB[j];
                constexpr int cw = (w + 7) / 8;
                float ms = rmg[-cw];
                if constexpr ((w & 7) != 0) ms = fminf(ms, rmg[-cw + 1]);
                if (M8 - ms >= thr * csqrt(w)) bits |= 1u << j;
            });
        }
        if constexpr (NL > 0) { // lane j: width j against the whole block (9 rows of 32 slots hold its starts)
            const float Emax = warp_max(M8);
            const float *rl = rm32 + (T.g0 >> 2) + T.rr; // row of the width's first start, in the upper copy
            float mn = S4_INF;
#pragma unroll
            for (int q = 0; q < 9; ++q) mn = fminf(mn, rl[q]);
            if (is_large && (Emax - mn) >= thr * sqw_lane) bits |= 1u << lane;
        }
    }

    // ---- widths <= SDIR: every cell, from the lane's samples and the few before them
    float Wn[24];
#pragma unroll
    for (int i = 0; i < 8; ++i) Wn[16 + i] = p8[i];
    const int g1 = wrapG(g - 1);
    if constexpr (ND > 0) {
        {
            const float4 d = *reinterpret_cast<const float4 *>(ring + PL1 + 4 * g1);
            Wn[12] = d.x; Wn[13] = d.y; Wn[14] = d.z; Wn[15] = d.w;
            if constexpr (SDIR > 4) {
                const float4 c = *reinterpret_cast<const float4 *>(ring + 4 * g1);
                Wn[8] = c.x; Wn[9] = c.y; Wn[10] = c.z; Wn[11] = c.w;
            }
        }
        float vb = -S4_INF;
        sfor<0, ND>([&](auto q) {
            constexpr int w = W_TAB[class_idx(0, V(q))];
            float m = T.md[V(q)];
#pragma unroll
            for (int i = 0; i < 8; ++i) m = fmaxf(m, E[i] - Wn[16 + i - w]);
            T.md[V(q)] = m;
            vb = fmaxf(vb, m * (1.0f / csqrt(w)));
        });
        if constexpr (PRUNE) {
            vb = warp_max(vb);
            if (vb > -S4_INF) publish(T, sbest, vb * T.rsig, lane);
        }
    }

    // ---- the widths whose bound can reach S*: rare
    const unsigned any = PRUNE ? __reduce_or_sync(kFull, bits) : (class_mask(1) | class_mask(2) | class_mask(3));
    if (any) {
        if constexpr (NWN > 0) {
            if (any & class_mask(1)) {
                const int g2 = wrapG(g - 2);
                const float4 a = *reinterpret_cast<const float4 *>(ring + 4 * g2);
                const float4 b = *reinterpret_cast<const float4 *>(ring + PL1 + 4 * g2);
                const float4 c = *reinterpret_cast<const float4 *>(ring + 4 * g1);
                const float4 d = *reinterpret_cast<const float4 *>(ring + PL1 + 4 * g1);
                Wn[0] = a.x; Wn[1] = a.y; Wn[2] = a.z; Wn[3] = a.w; Wn[4] = b.x; Wn[5] = b.y; Wn[6] = b.z; Wn[7] = b.w;
                Wn[8] = c.x; Wn[9] = c.y; Wn[10] = c.z; Wn[11] = c.w; Wn[12] = d.x; Wn[13] = d.y; Wn[14] = d.z; Wn[15] = d.w;
                sfor<0, NWN>([&](auto q) {
                    constexpr int j = class_idx(1, V(q));
                    constexpr int w = W_TAB[j];
                    if (any & (1u << j)) {
                        float m = T.mw[V(q)];
#pragma unroll
                        for (int i = 0; i < 8; ++i) m = fmaxf(m, E[i] - Wn[16 + i - w]);
                        T.mw[V(q)] = m;
                        if constexpr (PRUNE) {
                            const float v = warp_max(m);
                            if (v > -S4_INF) publish(T, sbest, v * (1.0f / csqrt(w)) * T.rsig, lane);
                        }
                    }
                });
            }
        }
        if constexpr (NM > 0) {
            sfor<0, NM>([&](auto q) {
                constexpr int j = class_idx(2, V(q));
                constexpr int w = W_TAB[j];
                if (any & (1u << j)) {
                    const float m = fmaxf(T.mm[V(q)], eval_far<w>(ring, g, E));
                    T.mm[V(q)] = m;
                    if constexpr (PRUNE) {
                        const float v = warp_max(m);
                        if (v > -S4_INF) publish(T, sbest, v * (1.0f / csqrt(w)) * T.rsig, lane);
                    }
                }
            });
        }
        if constexpr (NL > 0) {
            sfor<0, NL>([&](auto q) {
                constexpr int j = class_idx(3, V(q));
                constexpr int w = W_TAB[j];
                if (any & (1u << j)) {
                    const float v = warp_max(eval_far<w>(ring, g, E));
                    if (lane == j) T.ML = fmaxf(T.ML, v);
                    if constexpr (PRUNE) {
                        if (v > -S4_INF) publish(T, sbest, v * (1.0f / csqrt(w)) * T.rsig, lane);
                    }
                }
            });
        }
    }
    if constexpr (PRUNE) { // the next block's threshold: what any warp of the CTA has found so far
        const float sb = __int_as_float(*reinterpret_cast<volatile int *>(sbest));
        T.sbest = fmaxf(T.sbest, sb);
        T.thr = T.sbest * T.sigma * 0.99998f;
    }
    __syncwarp();
}

// the prefix of one block exactly as search_block forms it (same operations in the same order): p8 in, P[t+1] out
template <bool INSIDE> __device__ __forceinline__ void prefix_block(float (&p8)[8], float mu, float &carry, int lane, int nv)
{
    float run = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float x = (INSIDE || i < nv) ? p8[i] - mu : 0.f;
        run += x;
        p8[i] = run;
    }
    float ex;
    {
        float a = __shfl_up_sync(kFull, run, 1);
        if (lane == 0) a = 0.f;
        const float y1 = __shfl_up_sync(kFull, a, 1), y2 = __shfl_up_sync(kFull, a, 2), y3 = __shfl_up_sync(kFull, a, 3);
        const float s4 = (a + (lane >= 1 ? y1 : 0.f)) + ((lane >= 2 ? y2 : 0.f) + (lane >= 3 ? y3 : 0.f));
        const float z1 = __shfl_up_sync(kFull, s4, 4), z2 = __shfl_up_sync(kFull, s4, 8), z3 = __shfl_up_sync(kFull, s4, 12);
        const float s16 = (s4 + (lane >= 4 ? z1 : 0.f)) + ((lane >= 8 ? z2 : 0.f) + (lane >= 12 ? z3 : 0.f));
        const float q = __shfl_up_sync(kFull, s16, 16);
        ex = s16 + (lane >= 16 ? q : 0.f);
    }
    const float base = carry + ex;
#pragma unroll
    for (int i = 0; i < 8; ++i) p8[i] += base;
    carry = __shfl_sync(kFull, p8[7], 31);
}

// shared memory: rings, 8-slot minima (twice), 32-slot minima (twice) | per-(pixel, trial) results
constexpr int kRingFloats = NWARP * (RINGF + 2 * NG + 2 * NR);
constexpr int NBLK = (NT + LB - 1) / LB;                 // blocks of the longest series
constexpr int kSmemFloats = kRingFloats + PXI * NWARP * 8 + PXI * NWARP * NBLK + PXI * NWARP * 2;

// sweep A of one pixel: group G's delays are immediates here, and only here
template <int G> __device__ __forceinline__ void sweep_a(const float *Wp, float *scr, int tid)
{
    constexpr int T_g = NT - DMAX_TAB[G * NWARP];      // longest series of the group (trials are sorted by dmax)
    constexpr int TA = (T_g + LB - 1) / LB * LB;       // sweep B reads whole blocks
    for (int t = SPT * tid; t < TA; t += SPT * NTHR) dedisperse<G>(Wp + t, scr + t); // (reads past NT stay inside the padded workspace)
}

template <int G0, int N> __device__ __forceinline__ void dispatch_a(int g, const float *Wp, float *scr, int tid)
{
    if constexpr (N == 1) {
        sweep_a<G0>(Wp, scr, tid);
    } else {
        if (g < G0 + N / 2) dispatch_a<G0, N / 2>(g, Wp, scr, tid);
        else dispatch_a<G0 + N / 2, N - N / 2>(g, Wp, scr, tid);
    }
}

// one work item: pixels lp0 .. lp0 + npx - 1 of the batch, DM group g.  Everything after sweep A is the same code for every group.
__device__ __forceinline__ void run_item(const Search4Params &P, float *smem, int lp0, int npx, int g)
{
    float *rings = smem;                         // [NWARP][RINGF]  P[t+1] at slot t mod H, two planes
    float *rm8s = rings + NWARP * RINGF;         // [NWARP][2 NG]   min of P over each 8-slot group, stored twice
    float *rm32s = rm8s + NWARP * 2 * NG;        // [NWARP][2 NR]   min of P over each 32-slot row, stored twice
    float *red = rm32s + NWARP * 2 * NR;         // [PXI][NWARP][8] per-(pixel, trial) results
    float *cb = red + PXI * NWARP * 8;           // [PXI][NWARP][NBLK] the prefix before every block (the tail restarts there)
    float *tl = cb + PXI * NWARP * NBLK;         // [PXI][NWARP][2] tail: partial arg-max per slice
    __shared__ int sbest[PXI];                   // best S/N of each pixel so far (float bits, >= 0)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int u = g * NWARP + warp;
    const bool has = u < NU && (NT - DMAX_TAB[u < NU ? u : NU - 1]) >= 1;
    const int T_k = has ? NT - DMAX_TAB[u] : 0;
    float *ring = rings + warp * RINGF;
    float *rm8 = rm8s + warp * 2 * NG;
    float *rm32 = rm32s + warp * 2 * NR;
    float *scr0 = P.scratch + (size_t)blockIdx.x * PXI * NWARP * (size_t)DPITCH;

    // ================= sweep A: dedispersion of every pixel of the item -> scratch (no barrier inside)
    if (tid < PXI) sbest[tid] = 0;
    for (int px = 0; px < npx; ++px)
        dispatch_a<0, NGRP>(g, P.W + (size_t)(lp0 + px) * NCHAN * (size_t)PITCH, scr0 + (size_t)px * NWARP * DPITCH, tid);
    __syncthreads(); // every D of the item is in the scratch, visible to the whole CTA

    // ================= sweep B: warp = trial, pixel after pixel, no CTA barrier
    const int wl = lane < NW ? W_TAB[lane] : 0;
    const bool is_large = wl > WMID;
    const float sqw_lane = sqrtf((float)wl);
    constexpr int WMAXS = []() { int m = 1; for (int j = 0; j < NW; ++j) m = (W_TAB[j] > m && W_TAB[j] < H) ? W_TAB[j] : m; return m; }();
    constexpr int INIT = ((WMAXS + 95) / 32) * 32 < H ? ((WMAXS + 95) / 32) * 32 : H;
    for (int px = 0; px < npx; ++px) {
        float bs = -S4_INF;
        int bj = -1;
        float mu = 0.f, sigma = 0.f, mu_b = 0.f;
        if (has) {
            const float *drow = scr0 + ((size_t)px * NWARP + warp) * DPITCH;
            // ---- a1, a3: exact mean and sigma of the series (one pass; D is centred on the first sample of every channel)
            float rsig;
            {
                float s1 = 0.f, s2 = 0.f, s1b = 0.f, s2b = 0.f;
                int i = 4 * lane;
                for (; i + 388 <= T_k; i += 512) { // four independent 16-byte loads in flight per lane
                    const float4 v0 = __ldcg(reinterpret_cast<const float4 *>(drow + i));
                    const float4 v1 = __ldcg(reinterpret_cast<const float4 *>(drow + i + 128));
                    const float4 v2 = __ldcg(reinterpret_cast<const float4 *>(drow + i + 256));
                    const float4 v3 = __ldcg(reinterpret_cast<const float4 *>(drow + i + 384));
                    s1 += (v0.x + v0.y) + (v0.z + v0.w); s1b += (v1.x + v1.y) + (v1.z + v1.w);
                    s1 += (v2.x + v2.y) + (v2.z + v2.w); s1b += (v3.x + v3.y) + (v3.z + v3.w);
                    s2 = fmaf(v0.x, v0.x, s2); s2 = fmaf(v0.y, v0.y, s2); s2 = fmaf(v0.z, v0.z, s2); s2 = fmaf(v0.w, v0.w, s2);
                    s2b = fmaf(v1.x, v1.x, s2b); s2b = fmaf(v1.y, v1.y, s2b); s2b = fmaf(v1.z, v1.z, s2b); s2b = fmaf(v1.w, v1.w, s2b);
                    s2 = fmaf(v2.x, v2.x, s2); s2 = fmaf(v2.y, v2.y, s2); s2 = fmaf(v2.z, v2.z, s2); s2 = fmaf(v2.w, v2.w, s2);
                    s2b = fmaf(v3.x, v3.x, s2b); s2b = fmaf(v3.y, v3.y, s2b); s2b = fmaf(v3.z, v3.z, s2b); s2b = fmaf(v3.w, v3.w, s2b);
                }
                for (; i < T_k; i += 128) {
                    const float4 v = __ldcg(reinterpret_cast<const float4 *>(drow + i));
                    const float e[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        if (i + q < T_k) { s1 += e[q]; s2 = fmaf(e[q], e[q], s2); }
                }
                s1 += s1b;
                s2 += s2b;
                s1 = warp_sum(s1);
                s2 = warp_sum(s2);
                const float invT = 1.f / (float)T_k;
                mu = s1 * invT;
                sigma = sqrtf(fmaxf(fmaf(-mu, mu, s2 * invT), 0.f));
                rsig = sigma > 0.f ? 1.f / sigma : 0.f;
            }
            // "before time 0": only the slots a start can reach from the first blocks need the +inf marker -- the last INIT
            // slots of the ring (widest width + the rows the bounds look at); the rest is written before it is read
            for (int i = NG - INIT / 8 + lane; i < NG; i += 32) { // both planes of the group; P[0] = 0 sits in the very last slot
                const float4 inf4 = make_float4(S4_INF, S4_INF, S4_INF, S4_INF);
                *reinterpret_cast<float4 *>(ring + 4 * i) = inf4;
                *reinterpret_cast<float4 *>(ring + PL1 + 4 * i) = (i == NG - 1) ? make_float4(S4_INF, S4_INF, S4_INF, 0.f) : inf4;
                const float v = (i == NG - 1) ? 0.f : S4_INF;
                rm8[i] = v; rm8[i + NG] = v;
            }
            for (int i = NR - INIT / 32 + lane; i < NR; i += 32) { const float v = (i == NR - 1) ? 0.f : S4_INF; rm32[i] = v; rm32[i + NR] = v; }
            __syncwarp();
            Trial T;
            T.ML = -S4_INF;
#pragma unroll
            for (int q = 0; q < (ND > 0 ? ND : 1); ++q) T.md[q] = -S4_INF;
#pragma unroll
            for (int q = 0; q < (NWN > 0 ? NWN : 1); ++q) T.mw[q] = -S4_INF;
#pragma unroll
            for (int q = 0; q < (NM > 0 ? NM : 1); ++q) T.mm[q] = -S4_INF;
            T.mu = mu; T.sigma = sigma; T.rsig = rsig;
            T.carry = 0.f; T.sbest = 0.f; T.thr = PRUNE ? 0.f : -S4_INF; T.g0 = 0;
            T.rr = is_large ? NR - (wl + 31) / 32 : 0; // first start row of a block = its first end row - ceil(w/32), upper copy of rm32
            const float *dp = drow + 8 * lane;
            float4 na = __ldcg(reinterpret_cast<const float4 *>(dp)), nb = __ldcg(reinterpret_cast<const float4 *>(dp) + 1);
            for (int t0 = 0; t0 < T_k; t0 += LB) {
                float p8[8] = {na.x, na.y, na.z, na.w, nb.x, nb.y, nb.z, nb.w};
                if (t0 + LB < T_k) { // the next block's samples travel while this one is searched
                    na = __ldcg(reinterpret_cast<const float4 *>(dp + t0 + LB));
                    nb = __ldcg(reinterpret_cast<const float4 *>(dp + t0 + LB) + 1);
                }
                if (lane == 0) cb[(px * NWARP + warp) * NBLK + t0 / LB] = T.carry;
                if (t0 + LB <= T_k) search_block<true>(T, p8, ring, rm8, rm32, &sbest[px], lane, t0, T_k, sqw_lane, is_large);
                else search_block<false>(T, p8, ring, rm8, rm32, &sbest[px], lane, t0, T_k, sqw_lane, is_large);
                T.g0 = wrapG(T.g0 + LB / 8);
            }
            // ---- a6 (per trial): residual mean, normalise, best width
            const float delta = T.carry / (float)T_k; // P[T]/T: what float rounding left of the mean
            mu_b = T.mu;
            mu = T.mu + delta;
            float M = T.ML;
            sfor<0, ND>([&](auto q) {
                const float v = warp_max(T.md[V(q)]);
                if (lane == class_idx(0, V(q))) M = v;
            });
            sfor<0, NWN>([&](auto q) {
                const float v = warp_max(T.mw[V(q)]);
                if (lane == class_idx(1, V(q))) M = v;
            });
            sfor<0, NM>([&](auto q) {
                const float v = warp_max(T.mm[V(q)]);
                if (lane == class_idx(2, V(q))) M = v;
            });
            float S = -S4_INF;
            int jj = 0x7fffffff;
            if (lane < NW && M > -S4_INF) {
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
            float *r = red + (px * NWARP + warp) * 8;
            r[0] = bs;
            reinterpret_cast<int *>(r)[1] = (has && bj >= 0) ? K_OF_U[u] : -1;
            reinterpret_cast<int *>(r)[2] = bj;
            reinterpret_cast<int *>(r)[3] = u;
            r[4] = mu;     // the series' mean
            r[5] = sigma;
            r[7] = mu_b;   // the value sweep B centred the series on (the tail repeats its prefix)
        }
    }
    __syncthreads();

    // ================= tail: NWARP / npx warps per pixel: best trial, then the arg-max time -- the prefix of the winning series
    // once more (block by block from the saved carries, the same operations as sweep B: the same P bit for bit) into its
    // scratch row, and one scan of the winning width
    const int nsl = NWARP / npx;                 // warps (slices) per pixel
    const bool part = warp < npx * nsl;
    const int px = part ? warp / nsl : 0, sl = part ? warp - px * nsl : 0;
    const int p = P.p0 + lp0 + px;
    float s = -S4_INF, rmu = 0.f, rsg = 0.f, mu_b = 0.f;
    int k = -1, j = -1, uu = -1, wb = -1;
    if (part) { // (every slice of a pixel repeats this selection: lane w holds trial w's record)
        if (lane < NWARP) {
            const float *r = red + (px * NWARP + lane) * 8;
            s = r[0]; k = reinterpret_cast<const int *>(r)[1]; j = reinterpret_cast<const int *>(r)[2];
            uu = reinterpret_cast<const int *>(r)[3]; rmu = r[4]; rsg = r[5]; mu_b = r[7];
        }
        wb = (k >= 0) ? lane : -1;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float so = __shfl_xor_sync(kFull, s, o);
            const int ko = __shfl_xor_sync(kFull, k, o), jo = __shfl_xor_sync(kFull, j, o), wo = __shfl_xor_sync(kFull, wb, o);
            if (better(so, ko, jo, s, k, j)) { s = so; k = ko; j = jo; wb = wo; }
        }
        if (wb >= 0) {
            uu = __shfl_sync(kFull, uu, wb); rmu = __shfl_sync(kFull, rmu, wb); rsg = __shfl_sync(kFull, rsg, wb);
            mu_b = __shfl_sync(kFull, mu_b, wb);
        }
    }
    const int Tw = wb >= 0 ? NT - DMAX_TAB[uu] : 0, ww = wb >= 0 ? W_TAB[j] : 1;
    float *drow = scr0 + ((size_t)px * NWARP + (wb >= 0 ? wb : 0)) * DPITCH;
    if (part && wb >= 0) {
        const float *cbw = cb + (px * NWARP + wb) * NBLK;
        for (int t0 = sl * LB; t0 < Tw; t0 += nsl * LB) {
            float *dp = drow + t0 + 8 * lane;
            const float4 a = __ldcg(reinterpret_cast<const float4 *>(dp)), b = __ldcg(reinterpret_cast<const float4 *>(dp) + 1);
            float p8[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
            float carry = cbw[t0 / LB];
            if (t0 + LB <= Tw) prefix_block<true>(p8, mu_b, carry, lane, 8);
            else prefix_block<false>(p8, mu_b, carry, lane, Tw - t0 - 8 * lane);
            __stcg(reinterpret_cast<float4 *>(dp), make_float4(p8[0], p8[1], p8[2], p8[3]));
            __stcg(reinterpret_cast<float4 *>(dp) + 1, make_float4(p8[4], p8[5], p8[6], p8[7]));
        }
    }
    __syncthreads(); // the whole prefix series of every pixel's winner is in its scratch row
    if (part && wb >= 0) {
        float bv = -S4_INF;
        int bi = 0x7fffffff;
        const int last = Tw - ww; // starts 0..last; B = P[i+w] - P[i], P[i] at drow[i-1] (P[0] = 0)
        int i = sl * 32 + lane;
        const int step = nsl * 32;
        for (; i + 3 * step <= last; i += 4 * step) { // four starts per lane in flight
            float e[4], st[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                e[q] = __ldcg(drow + i + q * step + ww - 1);
                st[q] = (i + q * step == 0) ? 0.f : __ldcg(drow + i + q * step - 1);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float B = e[q] - st[q];
                if (B > bv) { bv = B; bi = i + q * step; }
            }
        }
        for (; i <= last; i += step) {
            const float B = __ldcg(drow + i + ww - 1) - (i == 0 ? 0.f : __ldcg(drow + i - 1));
            if (B > bv) { bv = B; bi = i; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float ov = __shfl_xor_sync(kFull, bv, o);
            const int oi = __shfl_xor_sync(kFull, bi, o);
            if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        if (lane == 0) { tl[(px * NWARP + sl) * 2] = bv; reinterpret_cast<int *>(tl)[(px * NWARP + sl) * 2 + 1] = bi; }
    }
    __syncthreads();
    if (part && sl == 0 && lane == 0) { // one thread per pixel: combine the slices, write the partial, take the ticket
        Partial4 out;
        out.snr = -S4_INF; out.k = -1; out.j = -1; out.t = -1; out.mu = 0.f; out.sigma = 0.f; out.u = -1; out.pad = 0;
        if (wb >= 0) {
            float bv = tl[(px * NWARP) * 2];
            int bi = reinterpret_cast<int *>(tl)[(px * NWARP) * 2 + 1];
            for (int q = 1; q < nsl; ++q) {
                const float ov = tl[(px * NWARP + q) * 2];
                const int oi = reinterpret_cast<int *>(tl)[(px * NWARP + q) * 2 + 1];
                if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
            }
            out.snr = s; out.k = k; out.j = j; out.t = bi; out.mu = rmu; out.sigma = rsg; out.u = uu;
        }
        P.partials[(size_t)p * NGRP + g] = out;
        __threadfence(); // the partial is visible before the ticket is taken
        const int prev = atomicAdd(P.counter + p, 1);
        if (prev == NGRP - 1) { // the pixel's last group: best partial -> outputs
            P.counter[p] = 0;   // ready for the next launch
            __threadfence();
            Partial4 b;
            b.snr = -S4_INF; b.k = -1; b.j = -1; b.t = -1; b.mu = 0.f; b.sigma = 0.f; b.u = -1; b.pad = 0;
            const int4 *pp = reinterpret_cast<const int4 *>(P.partials + (size_t)p * NGRP);
            for (int gg = 0; gg < NGRP; ++gg) {
                const int4 lo = __ldcg(pp + 2 * gg); // written by other CTAs: bypass L1
                const float snr = __int_as_float(lo.x);
                if (better(snr, lo.y, lo.z, b.snr, b.k, b.j)) { b.snr = snr; b.k = lo.y; b.j = lo.z; b.t = lo.w; }
            }
            P.snr_map[p] = b.k < 0 ? -S4_INF : b.snr;
            P.argmax[p] = b.k;
            P.argmax[(size_t)P.npix + p] = b.k < 0 ? -1 : J_OF_W[b.j];
            P.argmax[2 * (size_t)P.npix + p] = b.k < 0 ? -1 : b.t;
        }
    }
    __syncthreads(); // the next item reuses the scratch and the shared memory
}

} // namespace s4

extern "C" __global__ void __launch_bounds__(s4::NTHR, (NWARP < 16 ? 16 / NWARP : 1)) k_search4(const Search4Params P)
{
    extern __shared__ __align__(16) float smem[];
    const int noct = (P.npb + PXI - 1) / PXI;
    const int nitems = noct * s4::NGRP;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) { // consecutive CTAs share a pixel's rows in L2
        const int o = item / s4::NGRP;
        const int g = item - o * s4::NGRP;
        const int lp0 = o * PXI;
        s4::run_item(P, smem, lp0, (P.npb - lp0 < PXI) ? P.npb - lp0 : PXI, g);
    }
}

#endif
