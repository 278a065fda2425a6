// k_search4: the offline search kernel (steps a1..a6 of DESIGN.md), specialised per plan.
//
// Compiled at nsfrb_plan_prepare / the first nsfrb_search of a plan (NVRTC, sm_100a) behind a generated prologue:
//   NCHAN NU NW RS H PITCH DPITCH NT WMID SDIR LBA CHAIN RINGT SIDE PRUNE   integers
//                     RS raw-tile row stride, H prefix ring length (a multiple of 64), PITCH workspace row, DPITCH row of the
//                     dedispersed scratch, WMID/SDIR width classes (below), LBA x CHAIN the shape of the dedispersion sweep,
//                     RINGT the arg-max time comes out of the prefix ring (series that fit it), SIDE the kernel also moves
//                     the next pixel batch into the workspace, PRUNE = 0 switches the bounds off (every cell is evaluated)
//   D_TAB[NU][NCHAN]  delays of the unique trials (dmax ascending)   DMAX_TAB[NU]   K_OF_U[NU]
//   W_TAB[NW]         the usable widths, caller's order (NW <= 32)    J_OF_W[NW]     original width index
//
// Persistent CTAs (one per SM); a work item = one pixel x 16 trials, done in two sweeps over the time axis:
//   sweep A (CTA-wide, blocks of LBA samples)  cp.async stages the pixel's raw rows from the time-contiguous batch workspace;
//            differential dedispersion along the DM axis -- the first trial of a chain is the plain channel sum, every next one
//            adds (new - current) for the channels whose delay changed, the current value of every channel living in a
//            register, every shift an immediate; D goes to a per-CTA scratch (256-512 KB, L2-resident) and its sums S1, S2
//            stay in registers: after the sweep the exact mean and sigma of all 16 series are known (a1, a3)
//   sweep B (warp = trial, no CTA barrier; 8 consecutive samples per lane, blocks of 256)  x = D - mu, prefix by 8 serial
//            adds + one warp scan, P into the trial's ring (two interleaved planes of float4: every 128-bit access of a
//            warp is conflict-free), 8-sample minima beside it.  Because sigma is known, every boxcar is worth a known S/N and
//            a cell matters only if it can reach the best S/N the CTA has found so far (S*, shared by the 16 warps):
//              widths <= SDIR        every cell, from a 24-sample register window
//              widths SDIR+1..16     one bound for all of them (max of the lane's 8 ends - min of the 16 samples before),
//                                    then the register window for the widths whose own bound reaches S*
//              widths 17..WMID       per width: max of the 8 ends - min of the two 8-sample groups holding the starts;
//                                    the ring is read (three aligned float4) only if some lane's bound reaches S*
//              widths > WMID         lane j bounds width j for the whole block from 32-sample row minima; survivors as above
//            Every skipped cell is below its bound, hence below S* <= the CTA's final maximum: the maximum and its
//            (k, j, t) are exact.
//   end      S = (M - w delta)/(sigma sqrt(w)) per width, best width per trial, best trial per CTA; RINGT: the winning warp
//            finds the arg-max time in its ring; the last CTA of a pixel (ticket) reduces the pixel's partials -- and, for
//            series longer than the ring, rescans the winning series from the workspace (L2-hot) for the arg-max time.
// The workspace holds one BATCH of pixels; while an item is searched its CTA also moves its share of the next batch from the
// caller's [chan][time][pixel] cube into the other workspace buffer (SIDE), so the layout change needs no launch of its own.
#ifndef NSFRB_SEARCH_KERNEL_CUH
#define NSFRB_SEARCH_KERNEL_CUH

struct Partial4 { // layout of nsfrb::Partial (nsfrb_internal.h)
    float snr;
    int k, j, t; // t: window start of the maximum (RINGT), else -1
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
    float *scratch;     // [gridDim.x][16][DPITCH] dedispersed series of the item in flight
    // SIDE: the next batch, pixels [n0, n0 + nnb), goes from the caller's cube into Wn (nnb = 0: nothing to move)
    const float *cube;  // [NCHAN][NT][npix]
    float *Wn;          // [nnb][NCHAN][PITCH]
    int n0, nnb;
};

namespace s4 {

#define S4_INF __int_as_float(0x7f800000)
constexpr unsigned kFull = 0xffffffffu;
constexpr int NWARP = 16;  // trials (= warps) per CTA
constexpr int NTHR = NWARP * 32;
constexpr int LB = 256;    // samples per block of sweep B
constexpr int NR = H / 32; // ring rows of 32 slots
constexpr int NG = H / 8;  // ring groups of 8 slots (one lane's samples of a block)
constexpr int NGRP = (NU + NWARP - 1) / NWARP;
constexpr int PL1 = H / 2 + 16; // the ring's second plane: float4 chunk q of the series sits at (q & 1)*PL1 + 4*(q >> 1)
constexpr int RINGF = H + 16;
constexpr int NHALF = 16 / CHAIN;      // dedispersion chains per group
constexpr int ATHR = LBA * NHALF;      // threads of sweep A that dedisperse (<= NTHR)
constexpr int AWARPS = LBA / 32;       // warps per chain

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
__device__ __forceinline__ int wrapS(int s) // slot in (-H, 2H)
{
    if constexpr (HP2) return s & (H - 1);
    else return s < 0 ? s + H : (s >= H ? s - H : s);
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
__host__ __device__ constexpr int class_wmin(int c) { int m = 0x3fffffff; for (int j = 0; j < NW; ++j) if (wclass(W_TAB[j]) == c && W_TAB[j] < m) m = W_TAB[j]; return m; }
constexpr int ND = n_class(0), NWN = n_class(1), NM = n_class(2), NL = n_class(3);
__host__ __device__ constexpr float csqrt(int w) // sqrt(w), correctly rounded enough for a threshold (Newton in double)
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
__device__ __forceinline__ void cp_async16(float *dst, const float *src, int src_bytes)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async4(float *dst, const float *src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(src) : "memory");
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
}

__device__ __forceinline__ bool better(float s, int k, int j, float bs, int bk, int bj)
{
    if (k < 0) return false;
    if (bk < 0) return true;
    if (s != bs) return s > bs;
    if (k != bk) return k < bk;
    return j < bj;
}

// ---- SIDE: this item's share of the layout change of the next batch.  The 8*NGRP items of an aligned group of 8 pixels
// move the (channel, time) rows of the next batch's group of 8 pixels: member m takes rows [m*RPM, (m+1)*RPM) in steps of
// SROWS rows, one step per time block of sweep A.  A step reads its rows with cp.async (4-byte copies, lanes = 8 pixels x 4
// rows: whole 32-byte sectors) into a transposed tile [8][SROWS + 4]; one block later the tile goes out with lanes along time.
constexpr int SROWS = 256;
constexpr int TP = SROWS + 4; // tile pitch: 4 mod 32, so the transposing writes of a warp fall into 32 different banks
constexpr int NMEM = 8 * NGRP;
constexpr int ALLROWS = NCHAN * NT;
constexpr int RPM = (ALLROWS + NMEM - 1) / NMEM;
constexpr int NSTEP = (RPM + SROWS - 1) / SROWS;
constexpr int kSideFloats = SIDE ? 8 * TP : 0;

struct Side {
    int row0, row1; // this member's rows
    int pix8;       // first pixel of the group of 8, relative to the next batch
    bool on;
};

__device__ __forceinline__ void side_issue(const Search4Params &P, const Side &sd, float *tile, int step, int tid)
{
    if (!sd.on || step >= NSTEP) return;
    const int px = tid & 7, rs = tid >> 3; // 64 row slots x 8 pixels
    if (sd.pix8 + px >= P.nnb) return;
    const float *src = P.cube + (size_t)(P.n0 + sd.pix8 + px);
    float *dst = tile + px * TP + rs;
    const int r0 = sd.row0 + step * SROWS + rs;
#pragma unroll
    for (int k = 0; k < SROWS / 64; ++k) {
        const int r = r0 + 64 * k; // row = c*NT + t, which is also the row index of the cube
        if (r < sd.row1) cp_async4(dst + 64 * k, src + (size_t)r * (size_t)P.npix);
    }
}

__device__ __forceinline__ void side_store(const Search4Params &P, const Side &sd, const float *tile, int step, int tid)
{
    if (!sd.on || step < 0 || step >= NSTEP) return;
    const int px = tid >> 6, rs = tid & 63; // lanes along time
    if (sd.pix8 + px >= P.nnb) return;
    const size_t gp = (size_t)(P.n0 + sd.pix8 + px);
    float *dst = P.Wn + (size_t)(sd.pix8 + px) * NCHAN * (size_t)PITCH;
    const int r0 = sd.row0 + step * SROWS + rs;
#pragma unroll
    for (int k = 0; k < SROWS / 64; ++k) {
        const int r = r0 + 64 * k;
        if (r < sd.row1) {
            const int c = r / NT, t = r - c * NT;
            const float base = __ldg(P.cube + (size_t)c * NT * (size_t)P.npix + gp); // I[c][0][p], as k_transpose removes it
            dst[(size_t)c * PITCH + t] = tile[px * TP + rs + 64 * k] - base;
        }
    }
}

// ---- sweep A: differential dedispersion of sample t for CHAIN consecutive trials of group G starting at trial FIRST.
// rt = raw + (t - t0); dst = scratch + FIRST*DPITCH + t; s1/s2: the chain's running sums of D and D^2 over valid samples.
template <int G, int FIRST, bool MASK>
__device__ __forceinline__ void dedisperse(const float *__restrict__ rt, float *__restrict__ dst, int t, float (&s1)[CHAIN], float (&s2)[CHAIN])
{
    float cur[NCHAN];
    float acc = 0.f;
    sfor<0, CHAIN>([&](auto s) {
        constexpr int u = G * NWARP + FIRST + V(s);
        if constexpr (u < NU) {
            if constexpr (V(s) == 0) {
                float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
                sfor<0, NCHAN>([&](auto c) {
                    const float v = rt[V(c) * RS + D_TAB[u][V(c)]];
                    cur[V(c)] = v;
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
                        const float nv = rt[V(c) * RS + D_TAB[u][V(c)]];
                        const float v = nv - cur[V(c)];
                        cur[V(c)] = nv;
                        if constexpr ((V(c) & 1) == 0) a0 += v; else a1 += v;
                    }
                });
                acc += a0 + a1;
            }
            dst[V(s) * DPITCH] = acc;
            if (!MASK || t < NT - DMAX_TAB[u]) {
                s1[V(s)] += acc;
                s2[V(s)] = fmaf(acc, acc, s2[V(s)]);
            }
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
    float sbest;                 // the CTA's best S/N as this warp last saw it
    int g0, rr;                  // ring group of lane 0 in this block; ring row of the first start of the lane's large width
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
            if ((lane & 3) == 0) rm32[g >> 2] = lmin;
        }
    }
    __syncwarp();

    // the threshold in prefix units: a cell of width w matters only if B >= S* sigma sqrt(w) (a hair below, for rounding)
    if constexpr (PRUNE) {
        const float sb = __int_as_float(*reinterpret_cast<volatile int *>(sbest));
        T.sbest = fmaxf(T.sbest, sb);
    }
    float thr = PRUNE ? T.sbest * T.sigma * 0.99998f : -S4_INF;
    const float *rmg = rm8 + g + NG;

    // ---- widths <= 16 from a 24-sample register window
    if constexpr (ND + NWN > 0) {
        float Wn[24];
#pragma unroll
        for (int i = 0; i < 8; ++i) Wn[16 + i] = p8[i];
        {
            const int g1 = wrapG(g - 1), g2 = wrapG(g - 2);
            const float4 c = *reinterpret_cast<const float4 *>(ring + 4 * g1);
            const float4 d = *reinterpret_cast<const float4 *>(ring + PL1 + 4 * g1);
            Wn[8] = c.x; Wn[9] = c.y; Wn[10] = c.z; Wn[11] = c.w; Wn[12] = d.x; Wn[13] = d.y; Wn[14] = d.z; Wn[15] = d.w;
            constexpr int wneed = []() { int m = 0; for (int j = 0; j < NW; ++j) if (W_TAB[j] <= 16 && W_TAB[j] > m) m = W_TAB[j]; return m; }();
            if constexpr (wneed > 8) {
                const float4 a = *reinterpret_cast<const float4 *>(ring + 4 * g2);
                const float4 b = *reinterpret_cast<const float4 *>(ring + PL1 + 4 * g2);
                Wn[0] = a.x; Wn[1] = a.y; Wn[2] = a.z; Wn[3] = a.w; Wn[4] = b.x; Wn[5] = b.y; Wn[6] = b.z; Wn[7] = b.w;
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) Wn[i] = 0.f;
            }
        }
        if constexpr (ND > 0) {
            float vb = -S4_INF; // best direct cell so far, in units of sigma sqrt(w)... times sigma
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
                thr = T.sbest * T.sigma * 0.99998f;
            }
        }
        if constexpr (NWN > 0) {
            // one bound for all window widths: their starts lie in the 16 samples before the lane's first end and in
            // the lane's own group
            const float bnd = M8 - fminf(fminf(rmg[-2], rmg[-1]), m8own);
            constexpr float sq_min = csqrt(class_wmin(1));
            if (__any_sync(kFull, bnd >= thr * sq_min)) {
                float vb = -S4_INF;
                sfor<0, NWN>([&](auto q) {
                    constexpr int w = W_TAB[class_idx(1, V(q))];
                    float m = T.mw[V(q)];
#pragma unroll
                    for (int i = 0; i < 8; ++i) m = fmaxf(m, E[i] - Wn[16 + i - w]);
                    T.mw[V(q)] = m;
                    vb = fmaxf(vb, m * (1.0f / csqrt(w)));
                });
                if constexpr (PRUNE) {
                    vb = warp_max(vb);
                    if (vb > -S4_INF) publish(T, sbest, vb * T.rsig, lane);
                    thr = T.sbest * T.sigma * 0.99998f;
                }
            }
        }
    }
    // ---- widths 17..WMID: bound from the minima of the two 8-slot groups that hold the starts of the lane's 8 ends
    if constexpr (NM > 0) {
        sfor<0, NM>([&](auto q) {
            constexpr int w = W_TAB[class_idx(2, V(q))];
            constexpr int cw = (w + 7) / 8; // first start slot 8g - w lies in group g - cw
            float ms = rmg[-cw];
            if constexpr ((w & 7) != 0) ms = fminf(ms, rmg[-cw + 1]);
            if (__any_sync(kFull, M8 - ms >= thr * csqrt(w))) {
                const float m = fmaxf(T.mm[V(q)], eval_far<w>(ring, g, E));
                T.mm[V(q)] = m;
                if constexpr (PRUNE) {
                    const float vb = warp_max(m);
                    if (vb > -S4_INF) publish(T, sbest, vb * (1.0f / csqrt(w)) * T.rsig, lane);
                    thr = T.sbest * T.sigma * 0.99998f;
                }
            }
        });
    }
    // ---- widths > WMID: lane j bounds width j for the whole block: max of the block's ends - min over the 9 rows of 32
    //      slots that hold its starts; the widths that survive are evaluated like the mid widths
    if constexpr (NL > 0) {
        const float Emax = warp_max(M8);
        bool surv = false;
        if (is_large) {
            float mn = S4_INF;
            int r = T.rr;
#pragma unroll
            for (int q = 0; q < 9; ++q) {
                mn = fminf(mn, rm32[r]);
                r = wrapR(r + 1);
            }
            surv = (Emax - mn) >= thr * sqw_lane;
        }
        const unsigned mask = __ballot_sync(kFull, surv);
        if (mask) {
            sfor<0, NL>([&](auto q) {
                constexpr int j = class_idx(3, V(q));
                constexpr int w = W_TAB[j];
                if (mask & (1u << j)) {
                    const float v = warp_max(eval_far<w>(ring, g, E));
                    if (lane == j) T.ML = fmaxf(T.ML, v);
                    if constexpr (PRUNE) {
                        if (v > -S4_INF) publish(T, sbest, v * (1.0f / csqrt(w)) * T.rsig, lane);
                    }
                }
            });
        }
    }
    __syncwarp();
}

// ---- a6, last step of a pixel whose series are longer than the ring: best group, then the arg-max time by recomputing
// the winning series (L2-hot: the pixel's CTAs have just read it) with the mean/sigma the search found.
__device__ __forceinline__ void finalize_pixel(const Search4Params &P, float *fs, int p, const float *Wp)
{
    constexpr int PER = NTHR / 32;
    float *sc_f = fs + NT + 2;                        // [NTHR]
    int *sc_i = reinterpret_cast<int *>(sc_f + NTHR); // [NTHR]
    __shared__ Partial4 best;
    const int tid = threadIdx.x;
    if (tid == 0) {
        Partial4 b;
        b.snr = -S4_INF; b.k = -1; b.j = -1; b.t = -1; b.mu = 0.f; b.sigma = 0.f; b.u = -1; b.pad = 0;
        const int4 *pp = reinterpret_cast<const int4 *>(P.partials + (size_t)p * NGRP);
        for (int g = 0; g < NGRP; ++g) {
            const int4 lo = __ldcg(pp + 2 * g), hi = __ldcg(pp + 2 * g + 1); // written by other CTAs: bypass L1
            const float snr = __int_as_float(lo.x);
            if (better(snr, lo.y, lo.z, b.snr, b.k, b.j)) {
                b.snr = snr; b.k = lo.y; b.j = lo.z; b.t = lo.w;
                b.mu = __int_as_float(hi.x); b.sigma = __int_as_float(hi.y); b.u = hi.z; b.pad = hi.w;
            }
        }
        best = b;
    }
    __syncthreads();
    const Partial4 b = best;
    if (b.k < 0) {
        if (tid == 0) {
            P.snr_map[p] = -S4_INF;
            P.argmax[p] = -1; P.argmax[(size_t)P.npix + p] = -1; P.argmax[2 * (size_t)P.npix + p] = -1;
        }
        return;
    }
    if constexpr (RINGT) { // the CTA that found the maximum also found its time
        if (tid == 0) {
            P.snr_map[p] = b.snr;
            P.argmax[p] = b.k;
            P.argmax[(size_t)P.npix + p] = J_OF_W[b.j];
            P.argmax[2 * (size_t)P.npix + p] = b.t;
        }
        return;
    }
    const int w = W_TAB[b.j];
    const int n = NT - DMAX_TAB[b.u]; // samples [0, T): every start 0..T-w is a candidate
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
    float bv = -S4_INF;
    int bi = 0x7fffffff;
    for (int i = tid; i <= n - w; i += NTHR) {
        const float B = fs[i + w] - fs[i];
        if (B > bv) { bv = B; bi = i; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(kFull, bv, o);
        const int oi = __shfl_xor_sync(kFull, bi, o);
        if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    if ((tid & 31) == 0) { sc_f[tid >> 5] = bv; sc_i[tid >> 5] = bi; }
    __syncthreads();
    if (tid == 0) {
        for (int q = 1; q < NWARP; ++q)
            if (sc_f[q] > bv || (sc_f[q] == bv && sc_i[q] < bi)) { bv = sc_f[q]; bi = sc_i[q]; }
        const float S = b.sigma > 0.f ? bv / (b.sigma * sqrtf((float)w)) : 0.f;
        P.snr_map[p] = S;
        P.argmax[p] = b.k;
        P.argmax[(size_t)P.npix + p] = J_OF_W[b.j];
        P.argmax[2 * (size_t)P.npix + p] = bi;
    }
}

// shared memory: [raw tile of sweep A | rings, 8-slot minima (twice), 32-slot minima of sweep B] red, statistics, side tile
constexpr int kRawFloats = NCHAN * RS + 4;
constexpr int kRingFloats = NWARP * (RINGF + 2 * NG + NR);
constexpr int kStatFloats = NWARP * 2 * CHAIN + NWARP * 4; // per-warp partial sums of sweep A; mu, sigma, 1/sigma per trial
constexpr int kSmemFloats = kRawFloats + kRingFloats + NWARP * 8 + kStatFloats + kSideFloats;

template <int G> __device__ __forceinline__ void run_group(const Search4Params &P, float *smem, int lp)
{
    float *raw = smem;                           // [NCHAN][RS] (+4 pad)
    float *rings = raw + kRawFloats;             // [NWARP][RINGF]  P[t+1] at slot t mod H, two planes
    float *rm8s = rings + NWARP * RINGF;         // [NWARP][2 NG]   min of P over each 8-slot group, stored twice
    float *rm32s = rm8s + NWARP * 2 * NG;        // [NWARP][NR]     min of P over each 32-slot row
    float *red = rm32s + NWARP * NR;             // [NWARP][8]      per-trial results
    float *part = red + NWARP * 8;               // [NWARP][2 CHAIN] sweep A: per-warp sums
    float *stat = part + NWARP * 2 * CHAIN;      // [NWARP][4]      mu, sigma, 1/sigma, -
    float *tile = stat + NWARP * 4;              // [8][TP]         SIDE: transposing tile of the layout change
    __shared__ int sbest;                        // best S/N of the CTA so far (float bits, >= 0)
    __shared__ int is_last;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int p = P.p0 + lp;
    const int u = G * NWARP + warp;
    const bool has = u < NU && (NT - DMAX_TAB[u < NU ? u : NU - 1]) >= 1;
    const int T_k = has ? NT - DMAX_TAB[u] : 0;
    float *ring = rings + warp * RINGF;
    float *rm8 = rm8s + warp * 2 * NG;
    float *rm32 = rm32s + warp * NR;

    // group facts (static): the largest delay and the longest series
    constexpr int ulast = (G * NWARP + NWARP - 1 < NU) ? G * NWARP + NWARP - 1 : NU - 1;
    constexpr int dmax_g = DMAX_TAB[ulast];       // trials are sorted by dmax
    constexpr int T_g = NT - DMAX_TAB[G * NWARP]; // longest series of the group
    constexpr int T_gmin = NT - dmax_g;           // shortest
    constexpr int rows4 = (LBA + dmax_g + 3) & ~3;

    Side sd;
    sd.on = false; sd.row0 = 0; sd.row1 = 0; sd.pix8 = 0;
    if constexpr (SIDE) {
        const int m = (lp & 7) * NGRP + G;
        sd.pix8 = lp & ~7;
        sd.on = P.nnb > 0 && sd.pix8 < P.nnb;
        sd.row0 = m * RPM;
        sd.row1 = sd.row0 + RPM < ALLROWS ? sd.row0 + RPM : ALLROWS;
    }

    // ================= sweep A: dedispersion -> scratch, sums of D and D^2
    const float *Wp = P.W + (size_t)lp * NCHAN * (size_t)PITCH;
    float *scr = P.scratch + (size_t)blockIdx.x * NWARP * (size_t)DPITCH;
    if (tid == 0) sbest = 0;
    if (T_g > 0) issue_raw<rows4>(Wp, raw, 0, warp, lane);
    if constexpr (SIDE) side_issue(P, sd, tile, 0, tid);
    cp_async_commit();
    {
        float s1[CHAIN], s2[CHAIN];
#pragma unroll
        for (int i = 0; i < CHAIN; ++i) { s1[i] = 0.f; s2[i] = 0.f; }
        const int half = tid / LBA, tl = tid - half * LBA; // (half < NHALF for the dedispersing threads)
        int step = 0; // SIDE: the step whose rows are in flight
        for (int t0 = 0; t0 < T_g; t0 += LBA) {
            cp_async_wait_all();
            __syncthreads(); // raw(b) and the side tile landed
            if constexpr (SIDE) side_store(P, sd, tile, step, tid);
            if (tid < ATHR) {
                const float *rt = raw + tl;
                float *dst = scr + t0 + tl;
                const bool inside = t0 + LBA <= T_gmin;
                if constexpr (NHALF == 1) {
                    if (inside) dedisperse<G, 0, false>(rt, dst, t0 + tl, s1, s2);
                    else dedisperse<G, 0, true>(rt, dst, t0 + tl, s1, s2);
                } else {
                    if (half == 0) {
                        if (inside) dedisperse<G, 0, false>(rt, dst, t0 + tl, s1, s2);
                        else dedisperse<G, 0, true>(rt, dst, t0 + tl, s1, s2);
                    } else {
                        if (inside) dedisperse<G, CHAIN, false>(rt, dst + (size_t)CHAIN * DPITCH, t0 + tl, s1, s2);
                        else dedisperse<G, CHAIN, true>(rt, dst + (size_t)CHAIN * DPITCH, t0 + tl, s1, s2);
                    }
                }
            }
            __syncthreads(); // the raw tile and the side tile are free again
            if (t0 + LBA < T_g) issue_raw<rows4>(Wp, raw, t0 + LBA, warp, lane);
            if constexpr (SIDE) side_issue(P, sd, tile, ++step, tid);
            cp_async_commit();
        }
        if constexpr (SIDE) { // the steps the time blocks did not cover (short series, many rows)
            while (step < NSTEP) {
                cp_async_wait_all();
                __syncthreads();
                side_store(P, sd, tile, step, tid);
                __syncthreads();
                side_issue(P, sd, tile, ++step, tid);
                cp_async_commit();
            }
        }
        // per-warp sums -> shared memory -> one thread per trial
#pragma unroll
        for (int i = 0; i < CHAIN; ++i) {
            s1[i] = warp_sum(s1[i]);
            s2[i] = warp_sum(s2[i]);
        }
        if (lane == 0) {
#pragma unroll
            for (int i = 0; i < CHAIN; ++i) { part[warp * 2 * CHAIN + i] = s1[i]; part[warp * 2 * CHAIN + CHAIN + i] = s2[i]; }
        }
    }
    __syncthreads(); // (also: every D of the item is in the scratch, visible to the whole CTA)
    if (tid < NWARP) {
        const int h = tid / CHAIN, i = tid - h * CHAIN; // trial tid of the group: chain h, position i
        float S1 = 0.f, S2 = 0.f;
        for (int w = h * AWARPS; w < (h + 1) * AWARPS; ++w) { S1 += part[w * 2 * CHAIN + i]; S2 += part[w * 2 * CHAIN + CHAIN + i]; }
        const int uu = G * NWARP + tid;
        const int Tu = uu < NU ? NT - DMAX_TAB[uu < NU ? uu : NU - 1] : 0;
        float mu = 0.f, sg = 0.f;
        if (Tu >= 1) {
            const float invT = 1.f / (float)Tu;
            mu = S1 * invT;
            sg = sqrtf(fmaxf(fmaf(-mu, mu, S2 * invT), 0.f));
        }
        stat[tid * 4 + 0] = mu;
        stat[tid * 4 + 1] = sg;
        stat[tid * 4 + 2] = sg > 0.f ? 1.f / sg : 0.f;
    }
    // "before time 0": only the slots a start can reach from the first blocks need the +inf marker -- the last INIT slots
    // of the ring (widest width + the rows the bounds look at); the rest is written before it is read
    constexpr int WMAXS = []() { int m = 1; for (int j = 0; j < NW; ++j) m = (W_TAB[j] > m && W_TAB[j] < H) ? W_TAB[j] : m; return m; }();
    constexpr int INIT = ((WMAXS + 95) / 32) * 32 < H ? ((WMAXS + 95) / 32) * 32 : H;
    for (int s = H - INIT + lane; s < H; s += 32) ring[slot_addr(s)] = (s == H - 1) ? 0.f : S4_INF; // P[0] = 0 at slot -1
    for (int i = NG - INIT / 8 + lane; i < NG; i += 32) { const float v = (i == NG - 1) ? 0.f : S4_INF; rm8[i] = v; rm8[i + NG] = v; }
    for (int i = NR - INIT / 32 + lane; i < NR; i += 32) rm32[i] = (i == NR - 1) ? 0.f : S4_INF;
    __syncthreads();

    // ================= sweep B: warp = trial, no CTA barrier
    const int wl = lane < NW ? W_TAB[lane] : 0;
    const bool is_large = wl > WMID;
    Trial T;
    T.ML = -S4_INF;
#pragma unroll
    for (int q = 0; q < (ND > 0 ? ND : 1); ++q) T.md[q] = -S4_INF;
#pragma unroll
    for (int q = 0; q < (NWN > 0 ? NWN : 1); ++q) T.mw[q] = -S4_INF;
#pragma unroll
    for (int q = 0; q < (NM > 0 ? NM : 1); ++q) T.mm[q] = -S4_INF;
    T.mu = stat[warp * 4 + 0]; T.sigma = stat[warp * 4 + 1]; T.rsig = stat[warp * 4 + 2];
    T.carry = 0.f; T.sbest = 0.f; T.g0 = 0;
    T.rr = ((-wl) >> 5) + NR; // ring row of the first start of block 0 (floor division)
    if (T.rr >= NR || T.rr < 0) T.rr = 0;
    const float sqw_lane = sqrtf((float)wl);
    if (has) {
        const float *dp = scr + (size_t)warp * DPITCH + 8 * lane;
        float4 na = __ldcg(reinterpret_cast<const float4 *>(dp)), nb = __ldcg(reinterpret_cast<const float4 *>(dp) + 1);
        for (int t0 = 0; t0 < T_k; t0 += LB) {
            float p8[8] = {na.x, na.y, na.z, na.w, nb.x, nb.y, nb.z, nb.w};
            if (t0 + LB < T_k) { // the next block's samples travel while this one is searched
                na = __ldcg(reinterpret_cast<const float4 *>(dp + t0 + LB));
                nb = __ldcg(reinterpret_cast<const float4 *>(dp + t0 + LB) + 1);
            }
            if (t0 + LB <= T_k) search_block<true>(T, p8, ring, rm8, rm32, &sbest, lane, t0, T_k, sqw_lane, is_large);
            else search_block<false>(T, p8, ring, rm8, rm32, &sbest, lane, t0, T_k, sqw_lane, is_large);
            T.g0 = wrapG(T.g0 + LB / 8);
            T.rr = wrapR(T.rr + LB / 32);
        }
    }

    // ---- a6 (per trial): residual mean, normalise, best width
    float bs = -S4_INF;
    int bj = -1;
    float mu = 0.f, sigma = 0.f;
    if (has) {
        const float delta = T.carry / (float)T_k; // P[T]/T: what float rounding left of the mean (sigma is unaffected at this size)
        sigma = T.sigma;
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
        red[warp * 8 + 0] = bs;
        reinterpret_cast<int *>(red)[warp * 8 + 1] = (has && bj >= 0) ? K_OF_U[u] : -1;
        reinterpret_cast<int *>(red)[warp * 8 + 2] = bj;
        reinterpret_cast<int *>(red)[warp * 8 + 3] = u;
        red[warp * 8 + 4] = mu;
        red[warp * 8 + 5] = sigma;
    }
    __syncthreads();
    // best trial of the CTA (every thread walks the 16 records: the winning warp has to know it won)
    Partial4 out;
    out.snr = -S4_INF; out.k = -1; out.j = -1; out.t = -1; out.mu = 0.f; out.sigma = 0.f; out.u = -1; out.pad = 0;
    int wbest = -1;
    for (int w = 0; w < NWARP; ++w) {
        const float s = red[w * 8 + 0];
        const int k = reinterpret_cast<int *>(red)[w * 8 + 1], j = reinterpret_cast<int *>(red)[w * 8 + 2];
        if (better(s, k, j, out.snr, out.k, out.j)) {
            out.snr = s; out.k = k; out.j = j; out.u = reinterpret_cast<int *>(red)[w * 8 + 3];
            out.mu = red[w * 8 + 4]; out.sigma = red[w * 8 + 5];
            wbest = w;
        }
    }
    if constexpr (RINGT) {
        // the whole prefix series of the winning trial is still in its ring: smallest start of the maximum
        if (warp == wbest) {
            const int w = W_TAB[out.j];
            float bv = -S4_INF;
            int bi = 0x7fffffff;
            for (int i = lane; i <= T_k - w; i += 32) { // B = P[i+w] - P[i]; P[i] sits in slot i-1 (P[0] = 0)
                const float B = ring[slot_addr(i + w - 1)] - (i == 0 ? 0.f : ring[slot_addr(i - 1)]);
                if (B > bv) { bv = B; bi = i; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const float ov = __shfl_xor_sync(kFull, bv, o);
                const int oi = __shfl_xor_sync(kFull, bi, o);
                if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
            }
            if (lane == 0) {
                out.t = bi;
                P.partials[(size_t)p * NGRP + G] = out;
            }
        } else if (wbest < 0 && tid == 0) {
            P.partials[(size_t)p * NGRP + G] = out;
        }
    } else {
        if (tid == 0) P.partials[(size_t)p * NGRP + G] = out;
    }
    __syncthreads(); // the partial is written (by lane 0 of the winning warp, or thread 0)
    if (tid == 0) {
        __threadfence(); // ... and visible before the ticket is taken
        const int prev = atomicAdd(P.counter + p, 1);
        is_last = (prev == NGRP - 1);
        if (is_last) P.counter[p] = 0; // ready for the next launch
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        finalize_pixel(P, smem, p, Wp);
    }
    __syncthreads(); // the next item reuses the shared memory
}

template <int G0, int N> __device__ __forceinline__ void dispatch(int g, const Search4Params &P, float *smem, int lp)
{
    if constexpr (N == 1) {
        run_group<G0>(P, smem, lp);
    } else {
        if (g < G0 + N / 2) dispatch<G0, N / 2>(g, P, smem, lp);
        else dispatch<G0 + N / 2, N - N / 2>(g, P, smem, lp);
    }
}

} // namespace s4

extern "C" __global__ void __launch_bounds__(s4::NTHR, 1) k_search4(const Search4Params P)
{
    extern __shared__ __align__(16) float smem[];
    const int nitems = P.npb * s4::NGRP;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) { // consecutive CTAs share a pixel's rows in L2
        const int lp = item / s4::NGRP;
        const int g = item - lp * s4::NGRP;
        s4::dispatch<0, s4::NGRP>(g, P, smem, lp);
    }
}

#endif
