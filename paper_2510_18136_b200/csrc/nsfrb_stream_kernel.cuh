// k_stream and k_stream_stats: the kernels of nsfrb_stream_push (steps a1..a6 of DESIGN.md 5.2) for sm_100a.
//
// This file is compiled AT PLAN TIME (NVRTC, sm_100a) behind a generated prologue that fixes the
// plan's constants -- NPIX, NCHAN, the delay table, the width list, the ring length, the tile shape --
// so every dedispersion shift is an immediate and every register array is statically indexed
// ("shift indices for each frequency channel [are] pre-computed and loaded onto the GPU
// to minimize latencies"; here they are compiled into the instruction stream).  `build()` also compiles
// it ahead of time with the BASELINE config-2 prologue as a build check.
//
// Prologue (nsfrb_stream.cu: make_prologue):
//   NPIX NCHAN NU KK GPC SEG TT NW CMAX NSUPER MINB ROWS PFD INCR LIGHT NW_ALL CUBES DHIST COARSE LRING GUARD   integers
//     (INCR: statistics kept by k_stream_stats; LIGHT: plain runs take a shortcut; DHIST: the march reads the ring of
//      dedispersed samples; COARSE: and its 8-row block sums; LRING, GUARD: ring length and guard rows; NW_ALL: length of the
//      caller's width list; CUBES = 1 compiles the cube outputs in)
//   D_TAB[NU][NCHAN]   integer delays d[u][c] of the unique trials, DM ascending
//   DMAX_TAB[NU]       dmax_u                 K_OF_U[NU]  lowest original dm index of the trial
//   W_TAB[NW]          widths, ascending      J_OF_W[NW]  original width index   RSQ_W[NW]  1/sqrt(width)
//
// Reverse frame (all modes).  Series u has T_u = len - dmax_u samples; count them back from the newest one, r = 1..T_u.
// With Q_u(r) = sum_{r'<=r} (D_u(r') - mu0_u) (suffix sums of the series), the boxcar of width w whose window
// excludes the newest i samples is B(i, w) = Q(i+w) - Q(i); rule S5 (only windows whose last raw sample arrived
// in this push) keeps exactly i in [0, chunk_nt) for every trial.  One backward march therefore needs, per
// (pixel, trial): Q (register), Q at the C ends (shared memory, Qe) and the running max per width (M: one width
// at a time in registers, the rest in an L2-resident workspace -- wide widths have disjoint start ranges) -- no
// prefix history, no P ring.  Lane = pixel; thread = 1 pixel x KK consecutive trials x 1 of SEG time segments; a
// tile is TT steps; tiles that touch a width's start range also evaluate its cells (a5).  End of march:
// S = (M + Off - w delta)/(sigma sqrt(w)), reduced over widths, trials and DM groups of the CTA (a6).
//
// DHIST = 1 (the default): k_stream_stats dedisperses every sample ONCE, when it enters the valid set, and stores
// D_u(t) in dh[pixel block][row][trial][32] at the row of raw sample t + dmax_u -- so the r-th sample from the end of
// EVERY series sits in row top - (r - 1) and all trials march in step, each in its own frame.  k_stream reads one
// float per (trial, step), KK*TT values one tile ahead; in the plain runs between start ranges it adds whole 8-row
// blocks from dh8 (COARSE) and the ragged rows at the two ends.  Nothing but the trial column depends on the DM
// group: ONE instance of the march serves all groups (the instruction supply was the limit with one per group).
//
// DHIST = 0 (raw-ring march): the ring holds raw samples, D_u(r) = sum_c R[c][(r-1) + dmax_u - d[u][c]].  The KK
// trials of a thread march together in the GROUP frame rg = r - delta_u, delta_u = DMAXG - dmax_u: there trial u
// reads s = (rg-1) + e[u][c], e[u][c] = DMAXG - d[u][c], so consecutive trials differ only in the channels whose
// delay differs (differential dedispersion), every trial of the group ends at the same group step, and the delta_u
// newest samples of trial u are covered by a masked lead-in.  The ring is [block][row][chan][32]: every load is one
// coalesced 128-byte segment; the thread holds the raw window of every channel in registers (TT new rows + a
// carried halo of span_c rows), forms D for its first trial as the plain channel sum and every next trial
// differentially (a2).  One template instance per DM group.
#ifndef NSFRB_STREAM_KERNEL_CUH
#define NSFRB_STREAM_KERNEL_CUH

struct SPartial { // per (pixel, slice): slice = pass * NSUPER + supergroup
    float snr;
    int k, j, t; // original dm index, original width index, window start relative to ring sample 0
};

struct StreamParams {
    const float *ring; // [pixel block][ROWS][NCHAN][32], baseline removed, every sample stored at slot and slot+L
    float *mu0;        // [NU][NPIX] provisional means (the previous push's exact means); updated
    SPartial *partials;
    int top_row; // row of the newest sample
    int len;     // valid raw samples in the ring
    int i0, C;   // this pass evaluates ends i in [i0, i0+C)
    int nslice, slice0;
    float *mws;         // running maxima  [pixel block][supergroup][GPC*KK][NW][32]  (global, L2-resident)
    int *aws;           // their end indices, same shape
    float *sws;         // segment totals S1, S2  [pixel block][supergroup][2][GPC*KK][SEG][32]
    int bound[9];       // segment q < SEG marches steps (bound[q], bound[q+1]], multiples of TT (SEG <= 8)
    // optional per-(trial, width) outputs (S/N and TOA kept for all pixels x widths x DMs), or null:
    float *snr_cube;    // [NDM_ALL][NW_ALL][NPIX] peak S/N of every (dm, width) over this push's windows
    int *toa_cube;      // same shape: its window start (absolute, t_offset added); -1 where no window exists
    float *sig_out;     // [NU][NPIX] this push's sigma of every unique trial (running-sigma mode), or null
    int t_offset;
    // INCR = 1: mean and sigma are kept incrementally by k_stream_stats (nsfrb_stream.cu); mu0 then holds the exact mean
    // rounded to float, dlt the remainder (exact mean - mu0) and rsig = 1/sigma (0 where sigma = 0), all [NU][NPIX];
    // the march stops after the last start range and accumulates no sum of squares
    const float *dlt;
    const float *rsig;
    // DHIST = 1: the dedispersed history dh[pixel block][ROWS][NU][32] -- D_u(t) of every unique trial at the row of raw sample
    // t + dmax_u (same slots and double mapping as the ring), written once per sample by k_stream_stats when the sample enters
    // the valid set.  The march then reads one value per (trial, step) instead of dedispersing NCHAN channels, and the r-th
    // sample from the end of every series sits in row top_row - (r - 1): all trials march in their own frames, in step.
    const float *dh;
    // COARSE = 1 (needs LRING % 8 == 0): dh8[pixel block][2 * LRING / 8][NU][32], the sums of the 8-row aligned blocks of dh (block
    // b = rows 8b .. 8b+7 of the ring's slot space, stored at b and b + LRING/8), written when a block's last row arrives.
    // A plain run of the march adds whole blocks and only the ragged rows at its two ends one by one.
    const float *dh8;
};

#ifndef DHIST
#define DHIST 0
#endif
#ifndef COARSE
#define COARSE 0
#endif

namespace sk {

#define kInf __int_as_float(0x7f800000)

template <int I> struct IC {
    static constexpr int v = I;
    constexpr operator int() const { return I; }
};
// the value of an IC<> lambda argument as a constant expression
#define V(x) (decltype(x)::v)
template <int I, int N, class F> __device__ __forceinline__ void sfor(F &&f)
{
    if constexpr (I < N) {
        f(IC<I>{});
        sfor<I + 1, N>(f);
    }
}

// compile-time tables of DM group G (KK consecutive unique trials; the last group is padded by
// repeating the last trial, whose results are discarded)
template <int G> struct GT {
    static __host__ __device__ constexpr int u(int kk) { return (G * KK + kk < NU) ? G * KK + kk : NU - 1; }
    static __host__ __device__ constexpr int dmaxg()
    {
        int m = DMAX_TAB[u(0)];
        for (int k = 1; k < KK; ++k) m = DMAX_TAB[u(k)] > m ? DMAX_TAB[u(k)] : m;
        return m;
    }
    static __host__ __device__ constexpr int e(int kk, int c) { return dmaxg() - D_TAB[u(kk)][c]; }
    // own step = group step + delta.  (DHIST: the history stores D_u(t) at the row of raw sample t + dmax_u, so the r-th
    // sample from the end of EVERY series sits in row top - (r - 1): each trial marches in its own frame, delta = 0)
    static __host__ __device__ constexpr int delta(int kk) { return DHIST ? 0 : dmaxg() - DMAX_TAB[u(kk)]; }
    static __host__ __device__ constexpr int dspread()
    {
        int m = 0;
        for (int k = 0; k < KK; ++k) m = delta(k) > m ? delta(k) : m;
        return m;
    }
    static __host__ __device__ constexpr int emin(int c)
    {
        int m = e(0, c);
        for (int k = 1; k < KK; ++k) m = e(k, c) < m ? e(k, c) : m;
        return m;
    }
    static __host__ __device__ constexpr int emax(int c)
    {
        int m = e(0, c);
        for (int k = 1; k < KK; ++k) m = e(k, c) > m ? e(k, c) : m;
        return m;
    }
    static __host__ __device__ constexpr int span(int c) { return emax(c) - emin(c); }
    static __host__ __device__ constexpr int coff(int c)
    {
        int s = 0;
        for (int i = 0; i < c; ++i) s += span(i);
        return s;
    }
    static __host__ __device__ constexpr int o(int kk, int c) { return e(kk, c) - emin(c); }
    static constexpr int CARRY = coff(NCHAN) > 0 ? coff(NCHAN) : 1;
};

constexpr int kThreads = 32 * GPC * SEG;
constexpr int CURN = DHIST ? KK * TT : NCHAN * TT; // values a thread holds for one tile: D of its trials, or the raw rows
constexpr int kTrialsPerCta = GPC * KK;

// shared memory: Qe[kTrialsPerCta][CMAX][32], the cross-group reduction scratch, and per (group, segment)
// the range of widths that segment evaluated.  Segment totals S1, S2 [kTrialsPerCta][SEG][32] go through
// the global workspace sws (written once per thread).
constexpr int kQeFloats = kTrialsPerCta * CMAX * 32;
constexpr int QPAD = DHIST ? TT * 32 : 0; // floats of padding before and after Qe (the branch-free partial tiles read up to TT - 1 rows outside)
constexpr int kSegFloats = kTrialsPerCta * SEG * 32;
constexpr int kRedFloats = GPC * 32 * 4;
constexpr int kRangeInts = GPC * SEG * 2;
constexpr int kSmemBytes = (kQeFloats + 2 * QPAD + kRedFloats + kRangeInts) * 4;

__device__ __forceinline__ float ldrow(const float *p) { return __ldg(p); }

template <int G> struct Worker {
    using T = GT<G>;
    const float *rp;  // &ring[block][top_row][0][lane]
    const float *rp0; // the same for lane 0
#if DHIST
    const float *dp, *dp0; // &dh[block][top_row][u0][lane]; the row's first float
    // One instance of the march serves every DM group: with the history nothing but the trial column depends on the group
    // (G = 0 is the only instantiation), so the warps of an SM share one copy of the code.
    int u0; // first trial of the thread
    static constexpr bool kFull = NSUPER * GPC * KK == NU; // no padding trial anywhere
    __device__ __forceinline__ int uof(int kk) const { return (kFull || u0 + kk < NU) ? u0 + kk : NU - 1; }
    __device__ __forceinline__ bool has(int kk) const { return kFull || u0 + kk < NU; }
    __device__ __forceinline__ int ubase() const { return u0; }
    __device__ __forceinline__ int col(int kk) const { return uof(kk) - u0; } // column of the trial relative to dp (a padding trial repeats the last one)
#else
    static __device__ __forceinline__ constexpr int uof(int kk) { return T::u(kk); }
    static __device__ __forceinline__ constexpr bool has(int kk) { return G * KK + kk < NU; }
    static __device__ __forceinline__ constexpr int ubase() { return G * KK; }
#endif
    float *qe;       // &Qe[gl*KK][0][lane]
    float *mg;       // &mws[block][gl*KK][0][lane]
    int *ag;         // &aws[block][gl*KK][0][lane]
    int i0, C, len;
    float carry[DHIST ? 1 : T::CARRY];
    float mu[KK], dmu[KK], Q[KK], S2[KK]; // mu: provisional means (mu[0] and the differences dmu are live in the loop)
    int ja, jb; // widths [ja, jb) can have cells in the current tile
    const int *wt; // W_TAB in shared memory: a __device__ table indexed at run time is a global load, and these lookups sit on
                   // the critical path of every tile
    // register cache of one width's running maxima (the rest live in mws/aws)
    int jc, jfirst, jseen;
    float mc[KK];
    int ac[KK];

    __device__ __forceinline__ void flush()
    {
        if (jc >= 0) {
            float *mj = mg + jc * 32;
            int *aj = ag + jc * 32;
            sfor<0, KK>([&](auto kk) {
                if (has(V(kk))) {
                    mj[V(kk) * NW * 32] = mc[V(kk)];
                    aj[V(kk) * NW * 32] = ac[V(kk)];
                }
            });
        }
    }
    __device__ __forceinline__ void fetch(int j)
    {
        flush();
        if (j > jseen) { // first visit (widths are visited in ascending order)
            sfor<0, KK>([&](auto kk) { mc[V(kk)] = -kInf; ac[V(kk)] = 0; });
            jseen = j;
            if (jfirst < 0) jfirst = j;
        } else {
            const float *mj = mg + j * 32;
            const int *aj = ag + j * 32;
            sfor<0, KK>([&](auto kk) {
                if (has(V(kk))) {
                    mc[V(kk)] = mj[V(kk) * NW * 32];
                    ac[V(kk)] = aj[V(kk) * NW * 32];
                }
            });
        }
        jc = j;
    }

    __device__ __forceinline__ void load_new(float (&buf)[CURN], int rb) const
    {
#if DHIST
        // steps rb+1 .. rb+TT  <=>  history rows top - (rb + tt), one 128-byte segment per (trial, step)
        const float *d = dp - (long long)rb * (NU * 32);
        sfor<0, KK>([&](auto kk) {
            sfor<0, TT>([&](auto tt) { buf[V(kk) * TT + V(tt)] = ldrow(d + (col(V(kk)) - V(tt) * NU) * 32); });
        });
#else
        const float *b = rp - (long long)rb * (NCHAN * 32);
        sfor<0, NCHAN>([&](auto c) {
            sfor<0, TT>([&](auto tt) {
                constexpr int off = (V(c) - (T::span(V(c)) + V(tt) + T::emin(V(c))) * NCHAN) * 32;
                buf[V(c) * TT + V(tt)] = ldrow(b + off);
            });
        });
#endif
    }
    // ask L2 for the TT raw rows (all channels: TT*NCHAN*128 contiguous bytes in the blocked ring) that the tile
    // PFD tiles ahead will need first -- one bulk prefetch, no registers held; the later loads hit L2
    __device__ __forceinline__ void prefetch_l2(int rb) const
    {
#if DHIST
        const float *dlo = dp0 - (long long)(rb + TT - 1) * (NU * 32); // oldest of the TT rows, trial 0, lane 0
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(dlo), "r"(TT * NU * 128) : "memory");
#else
        constexpr int emax_all = []() { int m = 0; for (int c = 0; c < NCHAN; ++c) m = T::emax(c) > m ? T::emax(c) : m; return m; }();
        const float *lo = rp0 - (long long)(rb + emax_all + TT - 1) * (NCHAN * 32); // oldest of the TT rows, channel 0, lane 0
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(lo), "r"(TT * NCHAN * 128) : "memory");
#endif
    }
    __device__ __forceinline__ void load_carry(int rb)
    {
#if !DHIST // (the history holds finished samples: no halo)
        const float *b = rp - (long long)rb * (NCHAN * 32);
        sfor<0, NCHAN>([&](auto c) {
            sfor<0, T::span(V(c))>([&](auto m) {
                constexpr int off = (V(c) - (V(m) + T::emin(V(c))) * NCHAN) * 32;
                carry[T::coff(V(c)) + V(m)] = ldrow(b + off);
            });
        });
#endif
    }


#if LIGHT && DHIST && COARSE
    const float *dv0; // &dh[block][GUARD][0][lane]: virtual row v (0 .. 2*LRING-1; v mod LRING = ring slot) is dv0 + v*NU*32
    const float *dq0; // &dh8[block][0][0][lane]: block row v >> 3
    int vtop;         // virtual row of the newest sample
    // acc[kk] += sum over the rows [va, vb] and [vc, vd] of (base[(v * NU + u(kk)) * 32] - cm[kk])   (warp-uniform bounds, either
    // range may be empty; RIF rows = 32 loads in flight per thread).  cm: the provisional mean (times 8 for block sums) -- every
    // value is centred BEFORE it is accumulated, as in a tile, so the sums stay small where the level is far from zero.
    static constexpr int RIF = KK >= 8 ? 4 : (KK >= 4 ? 8 : 16);
    __device__ __forceinline__ void sum_rows(const float *base, int va, int vb, int vc, int vd, float scale, float (&acc)[KK]) const
    {
        const int n1 = vb >= va ? vb - va + 1 : 0, n = n1 + (vd >= vc ? vd - vc + 1 : 0);
        float cm[KK];
        sfor<0, KK>([&](auto kk) { cm[V(kk)] = scale * mu[V(kk)]; });
        for (int i = 0; i < n; i += RIF) {
            float x[RIF][KK];
            sfor<0, RIF>([&](auto q) {
                const int idx = i + V(q);
                const bool ok = idx < n;
                const int v = idx < n1 ? va + idx : vc + (idx - n1);
                const float *p = base + (long long)v * (NU * 32);
                sfor<0, KK>([&](auto kk) { x[V(q)][V(kk)] = ok ? ldrow(p + col(V(kk)) * 32) - cm[V(kk)] : 0.f; });
            });
            sfor<0, KK>([&](auto kk) {
                float t[RIF];
                sfor<0, RIF>([&](auto q) { t[V(q)] = x[V(q)][V(kk)]; });
                sfor<0, RIF / 2>([&](auto q) { t[V(q)] += t[V(q) + RIF / 2]; });
                if constexpr (RIF >= 4) sfor<0, RIF / 4>([&](auto q) { t[V(q)] += t[V(q) + RIF / 4]; });
                if constexpr (RIF >= 8) sfor<0, RIF / 8>([&](auto q) { t[V(q)] += t[V(q) + RIF / 8]; });
                if constexpr (RIF >= 16) t[0] += t[1];
                acc[V(kk)] += t[0];
            });
        }
    }
    // ---- a plain run (no end stored, no start range met), steps rb0+1 .. rb_end: only the suffix sums move.  The first tile is
    // already in `cur`; of the rest, whole 8-row blocks come from dh8, the ragged rows at the two ends from dh.
    __device__ __forceinline__ void coarse_run(float (&cur)[CURN], int rb0, int rb_end, bool more, bool pf)
    {
        float acc[KK];
        sfor<0, KK>([&](auto kk) {
            float a0 = 0.f, a1 = 0.f;
            sfor<0, TT>([&](auto tt) {
                if constexpr ((V(tt) & 1) == 0) a0 += cur[V(kk) * TT + V(tt)] - mu[V(kk)]; else a1 += cur[V(kk) * TT + V(tt)] - mu[V(kk)];
            });
            acc[V(kk)] = a0 + a1;
        });
        if (more) load_new(cur, rb_end); // the tile after the run
        if (PFD > 0 && pf && more) {      // ... and the rows behind it, which a start range will want
            const float *plo = dp0 - (long long)(rb_end + 2 * TT + 8 - 1) * (NU * 32);
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(plo), "r"((TT + 8) * NU * 128) : "memory");
        }
        const int top = vtop - rb0 - TT, v_lo = vtop - (rb_end - 1); // rows [v_lo, top] remain (step r <-> row vtop - (r - 1))
        if (top >= v_lo) {
            const int bfirst = (v_lo + 7) >> 3, blast = ((top + 1) >> 3) - 1;
            if (blast >= bfirst) {
                sum_rows(dv0, 8 * (blast + 1), top, v_lo, 8 * bfirst - 1, 1.f, acc); // the ragged rows at both ends, in one go
                sum_rows(dq0, bfirst, blast, 0, -1, 8.f, acc);
            } else {
                sum_rows(dv0, v_lo, top, 0, -1, 1.f, acc);
            }
        }
        sfor<0, KK>([&](auto kk) { Q[V(kk)] += acc[V(kk)]; });
    }
#elif LIGHT && DHIST
    // ---- plain runs (no end stored, no start range met): only the suffix sums move, one history value per (trial, step)
    __device__ __forceinline__ void run_begin() {}
    __device__ __forceinline__ void run_end(float, int) {}
    __device__ __forceinline__ void light(float (&cur)[CURN], int rb, bool more, bool pf, float &)
    {
        float part[KK];
        sfor<0, KK>([&](auto kk) {
            float a0 = -(float)TT * mu[V(kk)], a1 = 0.f;
            sfor<0, TT>([&](auto tt) {
                if constexpr ((V(tt) & 1) == 0) a0 += cur[V(kk) * TT + V(tt)]; else a1 += cur[V(kk) * TT + V(tt)];
            });
            part[V(kk)] = a0 + a1;
        });
        if (more) load_new(cur, rb + TT);
        if (PFD > 0 && pf) prefetch_l2(rb + PFD * TT);
        sfor<0, KK>([&](auto kk) { Q[V(kk)] += part[V(kk)]; });
    }
#elif LIGHT
    // ---- plain runs (no end stored, no start range met): only the suffix sums move.  Over a run of n steps trial kk adds
    //   sum_c sum_{m = o(kk,c)}^{n-1+o(kk,c)} W_c[m]  =  sum_c sum_{m<n} W_c[m]  +  edge(kk) at the exit  -  edge(kk) at the entry,
    // W_c[m] the raw window of channel c counted from the run's first row and edge(kk) = sum_c sum_{m<o(kk,c)} W_c[m], the
    // part of the carried halo below the trial's offset.  The first term is common to the KK trials: a light tile adds
    // the TT rows that leave the window (NCHAN*TT adds for all trials together) instead of dedispersing every trial.
    template <int KKI> __device__ __forceinline__ float edge_of() const
    {
        float a0 = 0.f, a1 = 0.f;
        sfor<0, NCHAN>([&](auto c) {
            sfor<0, T::o(KKI, V(c))>([&](auto m) {
                if constexpr (((V(c) + V(m)) & 1) == 0) a0 += carry[T::coff(V(c)) + V(m)];
                else a1 += carry[T::coff(V(c)) + V(m)];
            });
        });
        return a0 + a1;
    }
    __device__ __forceinline__ void run_begin()
    {
        sfor<0, KK>([&](auto kk) { Q[V(kk)] -= edge_of<V(kk)>(); });
    }
    // g: sum of the rows that left, centred on mu[0] per step; n steps
    __device__ __forceinline__ void run_end(float g, int n)
    {
        const float fn = (float)n;
        float cd = 0.f; // mu[0] - mu[kk]
        sfor<0, KK>([&](auto kk) {
            if constexpr (V(kk) > 0) cd += dmu[V(kk)];
            Q[V(kk)] += (g + edge_of<V(kk)>()) + fn * cd;
        });
    }
    __device__ __forceinline__ void light(float (&cur)[CURN], int rb, bool more, bool pf, float &g)
    {
        auto Wn = [&](auto c, auto m) -> float {
            if constexpr (V(m) < T::span(V(c))) return carry[T::coff(V(c)) + V(m)];
            else return cur[V(c) * TT + (V(m) - T::span(V(c)))];
        };
        float a0 = -(float)TT * mu[0], a1 = 0.f, a2 = 0.f, a3 = 0.f;
        sfor<0, NCHAN>([&](auto c) {
            sfor<0, TT>([&](auto tt) {
                const float v = Wn(c, tt);
                constexpr int sel = (V(c) * TT + V(tt)) & 3;
                if constexpr (sel == 0) a0 += v; else if constexpr (sel == 1) a1 += v; else if constexpr (sel == 2) a2 += v; else a3 += v;
            });
        });
        sfor<0, NCHAN>([&](auto c) {
            sfor<0, T::span(V(c))>([&](auto m) { carry[T::coff(V(c)) + V(m)] = Wn(c, IC<V(m) + TT>{}); });
        });
        if (more) load_new(cur, rb + TT);
        if (PFD > 0 && pf) prefetch_l2(rb + PFD * TT);
        g += (a0 + a1) + (a2 + a3);
    }
#endif
    // One tile: group steps rb+1 .. rb+TT.  On entry cur holds the TT new rows of every channel; on exit
    // (if `more`) the rows of the next tile have been requested into the same registers.
    // `cells`: the tile stores ends or meets a start range (one code body serves plain and cell tiles: the
    // hot instruction footprint of an SM has to stay within the ~32 KB the instruction cache streams well)
    template <bool MASKED> __device__ __forceinline__ void tile(float (&cur)[CURN], int rb, bool more, bool pf, bool cells)
    {
        float Dv[KK][TT];
#if DHIST
        sfor<0, KK>([&](auto kk) {
            sfor<0, TT>([&](auto tt) { Dv[V(kk)][V(tt)] = cur[V(kk) * TT + V(tt)] - mu[V(kk)]; });
        });
#else
        auto Wn = [&](auto c, auto m) -> float {
            if constexpr (V(m) < T::span(V(c))) return carry[T::coff(V(c)) + V(m)];
            else return cur[V(c) * TT + (V(m) - T::span(V(c)))];
        };
        // a2: first trial = plain channel sum, every next one differentially
        sfor<0, KK>([&](auto kk) {
            if constexpr (V(kk) == 0) {
                sfor<0, TT>([&](auto tt) {
                    float a0 = -mu[0], a1 = 0.f; // centred on the provisional mean of trial 0
                    sfor<0, NCHAN>([&](auto c) {
                        const float v = Wn(c, IC<V(tt) + T::o(0, V(c))>{});
                        if constexpr ((V(c) & 1) == 0) a0 += v; else a1 += v;
                    });
                    Dv[0][V(tt)] = a0 + a1;
                });
            } else {
                sfor<0, TT>([&](auto tt) {
                    float a = dmu[V(kk)]; // mu0[kk-1] - mu0[kk]: keeps every trial centred on its own provisional mean
                    sfor<0, NCHAN>([&](auto c) {
                        if constexpr (T::o(V(kk), V(c)) != T::o(V(kk) - 1, V(c)))
                            a += Wn(c, IC<V(tt) + T::o(V(kk), V(c))>{}) - Wn(c, IC<V(tt) + T::o(V(kk) - 1, V(c))>{});
                    });
                    Dv[V(kk)][V(tt)] = Dv[V(kk) - 1][V(tt)] + a;
                });
            }
        });
        // carry the halo: next tile's element m is this tile's element m + TT
        // (in place, ascending m: element m + TT is read before it is overwritten)
        sfor<0, NCHAN>([&](auto c) {
            sfor<0, T::span(V(c))>([&](auto m) { carry[T::coff(V(c)) + V(m)] = Wn(c, IC<V(m) + TT>{}); });
        });
#endif
        if (more) load_new(cur, rb + TT); // rows of the next tile; their latency overlaps what follows
        if (PFD > 0 && pf) prefetch_l2(rb + PFD * TT);
        // a1, a3, a4: centred sample, suffix sum (left in Dv), sum of squares
        sfor<0, KK>([&](auto kk) {
            sfor<0, TT>([&](auto tt) {
                float x = Dv[V(kk)][V(tt)];
                if constexpr (MASKED) {
                    const int ro = rb + 1 + V(tt) + T::delta(V(kk)); // step in the trial's own frame
                    x = (ro >= 1 && ro <= len - DMAX_TAB[uof(V(kk))]) ? x : 0.f;
                }
                Q[V(kk)] += x;
#if !INCR
                S2[V(kk)] = fmaf(x, x, S2[V(kk)]);
#endif
                Dv[V(kk)][V(tt)] = Q[V(kk)];
            });
        });
        if (cells && rb < i0 + C) {
            // Q at the ends of this pass: Qe[ii] = Q(i0 + ii), own frame
            float *qb = qe + (rb + 1 - i0) * 32;
            sfor<0, KK>([&](auto kk) {
                if (has(V(kk)))
                    sfor<0, TT>([&](auto tt) {
                        const unsigned ii = (unsigned)(rb + 1 - i0 + V(tt) + T::delta(V(kk)));
                        if (ii < (unsigned)C) qb[(V(kk) * CMAX + V(tt) + T::delta(V(kk))) * 32] = Dv[V(kk)][V(tt)];
                    });
            });
        }
        if (cells) {
            // a5: widths whose start range [w+i0, w+i0+C-1] (own frame) meets this tile
            while (ja < NW && wt[ja] + i0 + C - 1 < rb + 1) ++ja;
            if (jb < ja) jb = ja;
            while (jb < NW && wt[jb] + i0 <= rb + TT + T::dspread()) ++jb;
            for (int j = ja; j < jb; ++j) {
                if (j != jc) fetch(j);
                const int ib = rb + 1 - wt[j] - i0; // end index (relative to i0) of group step rb+1 at delta = 0
                const float *qb = qe + ib * 32;        // &Qe[0][ib]: every access below is a static offset from it
                const bool inside = !MASKED && ib >= 0 && ib + TT - 1 + T::dspread() < C;
                if (inside) { // every cell of the tile is defined: no range checks
                    sfor<0, KK>([&](auto kk) {
                        if (has(V(kk)))
                            sfor<0, TT>([&](auto tt) {
                                const float v = Dv[V(kk)][V(tt)] - qb[(V(kk) * CMAX + V(tt) + T::delta(V(kk))) * 32];
                                if (v >= mc[V(kk)]) { mc[V(kk)] = v; ac[V(kk)] = ib + V(tt) + T::delta(V(kk)); }
                            });
                    });
                } else {
                    sfor<0, KK>([&](auto kk) {
                        if (has(V(kk)))
                            sfor<0, TT>([&](auto tt) {
                                const int ii = ib + V(tt) + T::delta(V(kk));
                                bool in = (unsigned)ii < (unsigned)C;
                                if constexpr (MASKED) {
                                    const int ro = rb + 1 + V(tt) + T::delta(V(kk));
                                    in = in && ro >= 1 && ro <= len - DMAX_TAB[uof(V(kk))];
                                }
#if DHIST
                                // branch-free: an end outside [0, C) reads a neighbouring row of Qe (or its padding, QPAD rows on
                                // either side) and is replaced by -inf, which never beats a defined cell
                                const float d = Dv[V(kk)][V(tt)] - qb[(V(kk) * CMAX + V(tt)) * 32];
                                const float v = in ? d : -kInf;
                                if (v >= mc[V(kk)]) { mc[V(kk)] = v; ac[V(kk)] = ii; } // later step = earlier start
#else
                                if (in) {
                                    const float v = Dv[V(kk)][V(tt)] - qb[(V(kk) * CMAX + V(tt) + T::delta(V(kk))) * 32];
                                    if (v >= mc[V(kk)]) { mc[V(kk)] = v; ac[V(kk)] = ii; } // later step = earlier start
                                }
#endif
                            });
                    });
                }
            }
        }
    }
};

__device__ __forceinline__ void bar_named(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// (snr, k, j, t) ordering of O6: larger snr, then smaller original k, smaller original j, smaller t
__device__ __forceinline__ bool better(float s, int k, int j, int t, float bs, int bk, int bj, int bt)
{
    if (k < 0) return false;
    if (bk < 0) return true;
    if (s != bs) return s > bs;
    if (k != bk) return k < bk;
    if (j != bj) return j < bj;
    return t < bt;
}

template <int G>
__device__ __forceinline__ void run_group(const StreamParams &P, float *smem, const int *wtab, int gl, int seg, int lane, int pix, bool live, int u0 = 0)
{
    using T = GT<G>;
    float *Qe = smem + QPAD;
    float *red = Qe + kQeFloats + QPAD;
    float *S1s = P.sws + ((long long)blockIdx.x * NSUPER + blockIdx.y) * 2 * kSegFloats;
    float *S2s = S1s + kSegFloats;
    int *rng = reinterpret_cast<int *>(red + kRedFloats);

    Worker<G> w;
    w.wt = wtab;
#if DHIST
    w.u0 = u0;
#endif
    w.i0 = P.i0; w.C = P.C; w.len = P.len;
    w.rp0 = P.ring + ((long long)blockIdx.x * ROWS + P.top_row) * (NCHAN * 32);
    w.rp = w.rp0 + lane;
#if DHIST
    w.dp0 = P.dh + ((long long)blockIdx.x * ROWS + P.top_row) * (NU * 32);
    w.dp = w.dp0 + u0 * 32 + lane;
#if LIGHT && COARSE
    w.vtop = P.top_row - GUARD;
    w.dv0 = P.dh + ((long long)blockIdx.x * ROWS + GUARD) * (NU * 32) + u0 * 32 + lane;
    w.dq0 = P.dh8 + (long long)blockIdx.x * (2 * LRING / 8) * (NU * 32) + u0 * 32 + lane;
#endif
#endif
    w.qe = Qe + (gl * KK) * CMAX * 32 + lane;
    {
        const long long blk = ((long long)blockIdx.x * NSUPER + blockIdx.y) * kTrialsPerCta + gl * KK;
        w.mg = P.mws + blk * NW * 32 + lane;
        w.ag = P.aws + blk * NW * 32 + lane;
    }
    w.ja = 0; w.jb = 0; w.jc = -1; w.jfirst = -1; w.jseen = -1;
    sfor<0, KK>([&](auto kk) {
        w.mu[V(kk)] = P.mu0[(long long)w.uof(V(kk)) * NPIX + pix];
        w.Q[V(kk)] = 0.f;
        w.S2[V(kk)] = 0.f;
        w.dmu[V(kk)] = 0.f;
        w.mc[V(kk)] = -kInf;
        w.ac[V(kk)] = 0;
    });
    sfor<1, KK>([&](auto kk) { w.dmu[V(kk)] = w.mu[V(kk) - 1] - w.mu[V(kk)]; });
    if (seg == 0 && P.i0 == 0) sfor<0, KK>([&](auto kk) { w.qe[(V(kk) * CMAX) * 32] = 0.f; });

    // group frame: segment 0 starts with the masked lead-in that covers the newest delta_u samples
    constexpr int kLead = (T::dspread() + TT - 1) / TT * TT;
    const int r_begin = seg == 0 ? -kLead : P.bound[seg], r_end = P.bound[seg + 1];
#if DHIST
    int dmaxg = 0;
    sfor<0, KK>([&](auto kk) { dmaxg = DMAX_TAB[w.uof(V(kk))] > dmaxg ? DMAX_TAB[w.uof(V(kk))] : dmaxg; });
#else
    constexpr int dmaxg = T::dmaxg();
#endif
    const int r_fast_end = P.len - dmaxg; // last group step (valid for every trial of the group)
    const int qe_end = P.i0 + P.C;             // group steps < qe_end may store Qe (they lie in segment 0)
    const bool pf = gl == 0 && lane == 0; // the DM groups of a pixel block read the same rows: one thread prefetches
    bool synced = false;
    if (r_begin < r_end) {
        float cur[CURN];
        int rb = r_begin;
        w.load_carry(rb);
        w.load_new(cur, rb);
        int plain_until = r_begin; // exclusive
        // classify the tile at rb: does it store ends or meet a start range?  (also keeps the Qe barrier protocol)
        auto classify = [&]() -> bool {
            if (seg == 0 && !synced && rb >= qe_end) { // every Qe of this pass is written
                bar_named(1, kThreads);
                synced = true;
            }
            bool cells = rb >= plain_until; // tiles below plain_until are known to hold no end and no start
            if (cells) {
                cells = rb < qe_end;
                if (!cells) {
                    int ja = w.ja;
                    while (ja < NW && w.wt[ja] + P.i0 + P.C - 1 < rb + 1) ++ja;
                    w.ja = ja;
                    const int wnext = ja < NW ? w.wt[ja] + P.i0 - T::dspread() : 0x3fffffff; // first step of the next start range
                    cells = wnext <= rb + TT;
                    if (!cells) { // a plain run begins: nothing stays cached across it
                        plain_until = wnext - TT; // rb < plain_until  <=>  rb + TT < wnext
                        w.flush();
                        w.jc = -1;
                    }
                }
                if (cells && seg != 0 && !synced) { // Qe is complete once segment 0 has passed qe_end
                    bar_named(1, kThreads);
                    synced = true;
                }
            }
            return cells;
        };
        // three loops, so that the hot one holds a single tile body: masked lead-in (rb < 0), unmasked run, masked tail
        while (rb < r_end && rb < 0) {
            classify();
            w.template tile<true>(cur, rb, rb + TT < r_end, pf, true);
            rb += TT;
        }
        {
            const int fast_stop = r_end < r_fast_end - TT + 1 ? r_end : r_fast_end - TT + 1; // rb < fast_stop <=> tile fully valid
            while (rb < fast_stop) {
                const bool cells = classify();
#if LIGHT
                if (!cells) { // a plain run: up to the tile before the next start range (or the end of the unmasked part)
                    const int stop = plain_until < fast_stop ? plain_until : fast_stop;
#if DHIST && COARSE
                    {
                        const int nt = (stop - rb + TT - 1) / TT;
                        const int rb_end = rb + (nt > 1 ? nt : 1) * TT;
                        w.coarse_run(cur, rb, rb_end, rb_end < r_end, pf);
                        rb = rb_end;
                        continue;
                    }
#else
                    const int rb0 = rb;
                    float g = 0.f;
                    w.run_begin();
                    do {
                        w.light(cur, rb, rb + TT < r_end, pf, g);
                        rb += TT;
                    } while (rb < stop);
                    w.run_end(g, rb - rb0);
                    continue;
#endif
                }
#endif
                w.template tile<false>(cur, rb, rb + TT < r_end, pf, cells);
                rb += TT;
            }
        }
        while (rb < r_end) {
            classify();
            w.template tile<true>(cur, rb, rb + TT < r_end, pf, true);
            rb += TT;
        }
    }
    w.flush();
    if (!synced) bar_named(1, kThreads);

    // segment totals and the widths this segment evaluated
    sfor<0, KK>([&](auto kk) {
        S1s[((gl * KK + V(kk)) * SEG + seg) * 32 + lane] = w.Q[V(kk)];
#if !INCR
        S2s[((gl * KK + V(kk)) * SEG + seg) * 32 + lane] = w.S2[V(kk)];
#endif
    });
    if (lane == 0) {
        rng[(gl * SEG + seg) * 2 + 0] = w.jfirst;
        rng[(gl * SEG + seg) * 2 + 1] = w.jseen;
    }
    bar_named(2, kThreads);

    // a6: exact mean/variance, normalise, reduce over widths and trials (segment-0 threads)
    float bs = -kInf;
    int bk = -1, bj = -1, bt = -1;
    if (seg == 0) {
        // (a real loop over the thread's trials, tables indexed at run time: this code runs once per march, and
        // unrolled over KK trials x NW widths it was 150 KB of instructions fetched for a single pass)
#pragma unroll 1
        for (int kk = 0; kk < KK; ++kk) {
            const int u = w.ubase() + kk;
            if (u < NU) {
                const int Tk = P.len - DMAX_TAB[u];
                if (Tk >= 1) {
                    float off[SEG];
                    float s1 = 0.f, s2 = 0.f;
                    sfor<0, SEG>([&](auto q) {
                        off[V(q)] = s1;
                        s1 += S1s[((gl * KK + kk) * SEG + V(q)) * 32 + lane];
#if !INCR
                        s2 += S2s[((gl * KK + kk) * SEG + V(q)) * 32 + lane];
#endif
                    });
#if INCR
                    (void)s2;
                    const float delta = P.dlt[(long long)u * NPIX + pix];
                    const float rsig = P.rsig[(long long)u * NPIX + pix]; // 0 where sigma = 0 => S = 0 (definition)
#else
                    const float invT = 1.f / (float)Tk;
                    const float delta = s1 * invT;
                    const float var = fmaxf(fmaf(-delta, delta, s2 * invT), 0.f);
                    const float sigma = sqrtf(var);
                    const float rsig = sigma > 0.f ? 1.f / sigma : 0.f; // sigma = 0 => S = 0 (definition)
                    if (P.slice0 == 0 && live) P.mu0[(long long)u * NPIX + pix] += delta; // (still the value loaded into w.mu at the start)
#if CUBES
                    if (P.sig_out && P.slice0 == 0 && live) P.sig_out[(long long)u * NPIX + pix] = sigma;
#endif
#endif
                    // the running maxima of all widths of the trial come back from the workspace in one batch of
                    // independent loads (a width nobody visited holds stale values: read, then ignored) -- one round
                    // trip per trial instead of two dependent ones per (trial, width)
                    constexpr int JB = NW < 32 ? NW : 32; // widths per batch
                    sfor<0, (NW + JB - 1) / JB>([&](auto jb) {
                    constexpr int jlo = V(jb) * JB, jn = NW - jlo < JB ? NW - jlo : JB;
                    float mv[JB];
                    int av[JB];
                    sfor<0, jn>([&](auto j) {
                        mv[V(j)] = w.mg[(kk * NW + jlo + V(j)) * 32];
                        av[V(j)] = w.ag[(kk * NW + jlo + V(j)) * 32];
                    });
                    sfor<0, jn>([&](auto jc) {
                        constexpr int j = jlo + V(jc);
                        bool has = false; // did a segment evaluate the width (a width belongs to one segment)?
                        float offj = 0.f;
                        sfor<0, SEG>([&](auto q) {
                            const int j0 = rng[(gl * SEG + V(q)) * 2 + 0], j1 = rng[(gl * SEG + V(q)) * 2 + 1];
                            if (j0 >= 0 && j >= j0 && j <= j1) { has = true; offj = off[V(q)]; }
                        });
                        const float m = mv[V(jc)];
                        if (has && m > -kInf) {
                            constexpr int wj = W_TAB[j];
                            const float B = fmaf(-(float)wj, delta, m + offj);
                            const float S = (B * RSQ_W[j]) * rsig; // RSQ_W[j] = 1/sqrt(w_j), correctly rounded
                            const int ii = P.i0 + av[V(jc)];
                            const int t = Tk - ii - wj;
                            if (better(S, K_OF_U[u], J_OF_W[j], t, bs, bk, bj, bt)) { bs = S; bk = K_OF_U[u]; bj = J_OF_W[j]; bt = t; }
#if CUBES
                            if (P.snr_cube && live) { // cube entry: max over the passes of a push, ties to the smaller t
                                const long long ci = ((long long)K_OF_U[u] * NW_ALL + J_OF_W[j]) * NPIX + pix;
                                if (P.slice0 == 0 || S >= P.snr_cube[ci]) {
                                    P.snr_cube[ci] = S;
                                    P.toa_cube[ci] = (int)(((unsigned)P.t_offset + (unsigned)t) & 0x7fffffffu);
                                }
                            }
#endif
                        }
                    });
                    });
                }
            }
        }
        red[(gl * 32 + lane) * 4 + 0] = bs;
        reinterpret_cast<int *>(red)[(gl * 32 + lane) * 4 + 1] = bk;
        reinterpret_cast<int *>(red)[(gl * 32 + lane) * 4 + 2] = bj;
        reinterpret_cast<int *>(red)[(gl * 32 + lane) * 4 + 3] = bt;
    }
    // only the (group 0, segment 0) warp consumes the reduction scratch: the others arrive and leave
    if (!(seg == 0 && gl == 0)) {
        asm volatile("bar.arrive 3, %0;" ::"r"(kThreads) : "memory");
        return;
    }
    bar_named(3, kThreads);
    if (live) {
        sfor<1, GPC>([&](auto g2) {
            const float s = red[(V(g2) * 32 + lane) * 4 + 0];
            const int k = reinterpret_cast<int *>(red)[(V(g2) * 32 + lane) * 4 + 1];
            const int j = reinterpret_cast<int *>(red)[(V(g2) * 32 + lane) * 4 + 2];
            const int t = reinterpret_cast<int *>(red)[(V(g2) * 32 + lane) * 4 + 3];
            if (better(s, k, j, t, bs, bk, bj, bt)) { bs = s; bk = k; bj = j; bt = t; }
        });
        SPartial out;
        out.snr = bk < 0 ? -kInf : bs; out.k = bk; out.j = bk < 0 ? -1 : bj; out.t = bk < 0 ? -1 : bt;
        P.partials[(long long)pix * P.nslice + P.slice0 + blockIdx.y] = out;
    }
}

template <int G0, int N>
__device__ __forceinline__ void dispatch(int g, const StreamParams &P, float *smem, const int *wtab, int gl, int seg, int lane, int pix, bool live)
{
    if constexpr (N == 1) {
        run_group<G0>(P, smem, wtab, gl, seg, lane, pix, live);
    } else {
        if (g < G0 + N / 2) dispatch<G0, N / 2>(g, P, smem, wtab, gl, seg, lane, pix, live);
        else dispatch<G0 + N / 2, N - N / 2>(g, P, smem, wtab, gl, seg, lane, pix, live);
    }
}

} // namespace sk

extern "C" __global__ void __launch_bounds__(sk::kThreads, MINB) k_stream(const StreamParams P)
{
    extern __shared__ __align__(16) float smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int gl = warp / SEG, seg = warp - gl * SEG;
    // lanes past NPIX work on the last pixel (loads stay in bounds) and skip their stores
    int pix = blockIdx.x * 32 + lane;
    const bool live = pix < NPIX;
    if (!live) pix = NPIX - 1;
    const int g = blockIdx.y * GPC + gl; // DM group of this warp; NSUPER*GPC groups exist (the last may be padding)
    __shared__ int s_wtab[NW];
    for (int i = threadIdx.x; i < NW; i += sk::kThreads) s_wtab[i] = W_TAB[i];
    __syncthreads();
#if DHIST
    sk::run_group<0>(P, smem, s_wtab, gl, seg, lane, pix, live, g * KK);
#else
    sk::dispatch<0, NSUPER * GPC>(g, P, smem, s_wtab, gl, seg, lane, pix, live);
#endif
}

#if INCR
// a1, a3 kept incrementally: S1 = sum D_u, S2 = sum D_u^2 over the valid samples V_u = [lo, n - dmax_u) of every (unique
// trial u, pixel), in float64, carried from push to push.  The launch with add = 0 runs BEFORE the ring update and takes
// out the samples that leave V_u with this push (their raw rows are about to be overwritten); the one with add = 1 runs
// after it, puts in the samples that enter, and writes what k_stream needs: the mean (as a float, plus the remainder
// dlt = mean - float(mean)) and 1/sigma (population; 0 where sigma = 0).  A sample's D is formed from
// the same stored ring values in the same order when it enters and when it leaves, so the two contributions cancel to
// float64 rounding.  Lane = pixel, warp = trial; the trial's shifts are immediates.
struct StatsParams {
    const float *ring;
    double *s1, *s2;      // [NU][NPIX]
    float *mu, *dlt, *rsig, *sig_out;
    int row_lo;           // ring row that holds the raw sample of absolute index ring_lo
    int add, first, pad;
    long long ring_lo, lo_prev, n_prev, lo, n;
    float *dh;            // DHIST: the dedispersed history (see StreamParams), written by the add = 1 launch, read by add = 0
    float *dh8;           // COARSE: its 8-row block sums, written by the add = 1 launch
};

namespace sk {

// S1 += sum D, S2 += sum D^2 over cnt consecutive samples of trial U starting at ring pointer rp (lane = pixel).
// (A sample's D is the same expression wherever it falls in a range: entering, leaving and rebuilding must agree bit for bit.)
// dcol (DHIST, may be null): &dh[block][GUARD][U][lane]; the sample at ring slot `slot` is also stored there (both mappings).
template <int U> __device__ __forceinline__ void stats_range(const float *rp, int cnt, double &a1, double &a2, float *dcol = nullptr, int slot = 0)
{
    auto keep = [&](float Df) {
#if DHIST
        if (dcol) {
            dcol[(long long)slot * (NU * 32)] = Df;
            dcol[(long long)(slot + LRING) * (NU * 32)] = Df;
            slot = slot + 1 == LRING ? 0 : slot + 1;
        }
#endif
    };
    int i = cnt;
    for (; i >= 4; i -= 4, rp += 4 * NCHAN * 32) { // four samples per round: 4*NCHAN loads in flight
        float e[4][4] = {};
        sfor<0, 4>([&](auto q) {
            sfor<0, NCHAN>([&](auto c) { e[V(q)][V(c) & 3] += __ldg(rp + ((D_TAB[U][V(c)] + V(q)) * NCHAN + V(c)) * 32); });
        });
        sfor<0, 4>([&](auto q) {
            const float Df = (e[V(q)][0] + e[V(q)][1]) + (e[V(q)][2] + e[V(q)][3]);
            keep(Df);
            const double D = (double)Df;
            a1 += D;
            a2 = fma(D, D, a2);
        });
    }
    for (; i > 0; --i, rp += NCHAN * 32) {
        float e[4] = {0.f, 0.f, 0.f, 0.f};
        sfor<0, NCHAN>([&](auto c) { e[V(c) & 3] += __ldg(rp + (D_TAB[U][V(c)] * NCHAN + V(c)) * 32); });
        const float Df = (e[0] + e[1]) + (e[2] + e[3]);
        keep(Df);
        const double D = (double)Df;
        a1 += D;
        a2 = fma(D, D, a2);
    }
}
#if DHIST
// the same sums over cnt samples read back from the history (the float that was stored is the float that was added)
__device__ __forceinline__ void stats_history(const float *dcol, int slot, int cnt, double &a1, double &a2)
{
    const float *p = dcol + (long long)slot * (NU * 32); // slot < LRING, cnt <= LRING: the double mapping covers the run
    for (int i0 = 0; i0 < cnt; i0 += 32, p += 32 * NU * 32) { // one round trip per 32 samples (a push of 25: one)
        float d[32];
        sfor<0, 32>([&](auto q) { d[V(q)] = i0 + V(q) < cnt ? p[V(q) * NU * 32] : 0.f; }); // (plain loads: the fused launch stores to these rows afterwards)
        sfor<0, 32>([&](auto q) { const double D = (double)d[V(q)]; a1 += D; a2 = fma(D, D, a2); }); // (a padding zero adds nothing)
    }
}
#endif
// The rare paths (rebuild after a marked series, two-pass variance) over the whole valid set of trial u, with the shifts read
// from the table at run time: like everything in stats_trial but the loop over the entering samples, ONE copy of the code
// serves all trials (the eight trials of a CTA share the instruction cache).  Same expression and order as stats_range, so
// the same floats.
// centred = false: a1 += sum D, a2 += sum D^2;  centred = true: a2 += sum (D - centre)^2
__device__ __forceinline__ void stats_whole(int u, const float *rp, int cnt, bool centred, double centre, double &a1, double &a2)
{
    int off[NCHAN];
    sfor<0, NCHAN>([&](auto c) { off[V(c)] = ((int)D_TAB[u][V(c)] * NCHAN + V(c)) * 32; });
    for (int i = cnt; i > 0; --i, rp += NCHAN * 32) {
        float e[4] = {0.f, 0.f, 0.f, 0.f};
        sfor<0, NCHAN>([&](auto c) { e[V(c) & 3] += __ldg(rp + off[V(c)]); });
        const double D = (double)((e[0] + e[1]) + (e[2] + e[3]));
        if (centred) {
            const double x = D - centre;
            a2 = fma(x, x, a2);
        } else {
            a1 += D;
            a2 = fma(D, D, a2);
        }
    }
}

// the entering (or, without the history, leaving) samples of trial u: the only part compiled per trial (immediate shifts)
template <int U0, int N>
__device__ __forceinline__ void stats_range_of(int u, const float *rp, int cnt, double &a1, double &a2, float *dcol = nullptr, int slot = 0)
{
    if constexpr (N == 1) {
        stats_range<U0>(rp, cnt, a1, a2, dcol, slot);
    } else {
        if (u < U0 + N / 2) stats_range_of<U0, N / 2>(u, rp, cnt, a1, a2, dcol, slot);
        else stats_range_of<U0 + N / 2, N - N / 2>(u, rp, cnt, a1, a2, dcol, slot);
    }
}

__device__ __forceinline__ void stats_trial(const StatsParams &P, int U, int lane, int pix, bool live)
{
    // P.add: 0 = take out the samples that leave V_u, 1 = put in the ones that enter and publish, 2 = both (DHIST: the leaving
    // samples are read from the history, so nothing has to run before the ring update)
    const long long dm = DMAX_TAB[U];
    const bool do_rm = P.add != 1, do_add = P.add != 0;
    const long long b_prev = P.lo_prev > P.n_prev - dm ? P.lo_prev : P.n_prev - dm; // end of the previous valid set
    const long long la = P.lo_prev, lb = P.lo < b_prev ? P.lo : b_prev;             // leaving:  [la, lb)
    const long long ta = b_prev > P.lo ? b_prev : P.lo, tb = P.lo > P.n - dm ? P.lo : P.n - dm; // entering: [ta, tb)
    const float *rbase = P.ring + ((long long)blockIdx.x * ROWS + P.row_lo) * (NCHAN * 32) + lane; // sample ring_lo
    const long long o = (long long)U * NPIX + pix;
    const double kNaN = __longlong_as_double(0x7ff8000000000000LL);
#if DHIST
    float *dcol = P.dh + ((long long)blockIdx.x * ROWS + GUARD) * (NU * 32) + U * 32 + lane; // D_u(t) lives at the row of raw sample t + dmax_u
#endif
    double s1 = 0.0, s2 = 0.0; // the carried sums
    if (!P.first) { s1 = P.s1[o]; s2 = P.s2[o]; }
    if (do_rm && lb > la) {
        double a1 = 0.0, a2 = 0.0;
#if DHIST
        stats_history(dcol, (int)((la + dm) % LRING), (int)(lb - la), a1, a2);
#else
        stats_range_of<0, NU>(U, rbase + (la - P.ring_lo) * (NCHAN * 32), (int)(lb - la), a1, a2);
#endif
        // A leaving sample that dwarfs what stays behind (|D| beyond ~10^3 sigma sqrt(T)) has eaten the low bits of S2 when it
        // entered, and a non-finite one has destroyed the sums: mark the series (NaN); the add pass rebuilds it from the ring.
        const double r1 = s1 - a1, r2 = s2 - a2;
        const bool bad = !(a2 <= 1048576.0 * fabs(r2)) || !(fabs(r1) <= 1.7e308);
        s1 = bad ? kNaN : r1;
        s2 = bad ? kNaN : r2;
        if (!do_add && live) { P.s1[o] = s1; P.s2[o] = s2; }
    }
    if (!do_add) return;
    double a1 = 0.0, a2 = 0.0;
#if DHIST
    if (tb > ta) {
        stats_range_of<0, NU>(U, rbase + (ta - P.ring_lo) * (NCHAN * 32), (int)(tb - ta), a1, a2, dcol, (int)((ta + dm) % LRING));
#if COARSE
        { // the aligned rows [ra, rz) have just been written: every block whose last row is among them is complete
            const long long ra = ta + dm, rz = tb + dm;
            float *dcol8 = P.dh8 + (long long)blockIdx.x * (2 * LRING / 8) * (NU * 32) + U * 32 + lane;
            const long long b_hi = (rz - 8) >> 3;
            for (long long b0 = ra >> 3; b0 <= b_hi; b0 += 4) { // four blocks per round trip (a push of 25 samples completes 3 or 4)
                float d[4][8];
                int s8[4];
                sfor<0, 4>([&](auto j) {
                    const bool ok = b0 + V(j) <= b_hi;
                    s8[V(j)] = (int)((8 * (b0 + V(j))) % LRING); // slot of the block's first row (LRING % 8 == 0: the block does not wrap)
                    const float *r8 = dcol + (long long)s8[V(j)] * (NU * 32);
                    sfor<0, 8>([&](auto q) { d[V(j)][V(q)] = ok ? r8[V(q) * NU * 32] : 0.f; }); // (plain loads: some of these rows were stored above)
                });
                sfor<0, 4>([&](auto j) {
                    if (b0 + V(j) <= b_hi) {
                        const float E = ((d[V(j)][0] + d[V(j)][1]) + (d[V(j)][2] + d[V(j)][3])) + ((d[V(j)][4] + d[V(j)][5]) + (d[V(j)][6] + d[V(j)][7]));
                        dcol8[(long long)(s8[V(j)] >> 3) * (NU * 32)] = E;
                        dcol8[(long long)((s8[V(j)] >> 3) + LRING / 8) * (NU * 32)] = E;
                    }
                });
            }
        }
#endif
    }
#else
    stats_range_of<0, NU>(U, rbase + (ta - P.ring_lo) * (NCHAN * 32), (int)(tb - ta), a1, a2);
#endif
    const long long Tk = tb - P.lo; // tb = max(lo, n - dmax_u)
    bool rebuild = false;
    if (!P.first) {
        a1 += s1;
        a2 += s2;
        rebuild = !(fabs(a1) <= 1.7e308) || !(fabs(a2) <= 1.7e308); // marked, or poisoned by a non-finite sample
    }
    if (__any_sync(0xffffffffu, rebuild)) { // warp = one trial, lanes = pixels: the whole valid set once more (rare)
        double b1 = 0.0, b2 = 0.0;
        stats_whole(U, rbase + (P.lo - P.ring_lo) * (NCHAN * 32), (int)Tk, false, 0.0, b1, b2);
        if (rebuild) { a1 = b1; a2 = b2; }
    }
    float m = 0.f, dl = 0.f, rs = 0.f, sg = __int_as_float(0x7fc00000); // NaN sigma = "no valid sample yet"
    double mean = 0.0, var = 0.0;
    bool cancel = false;
    if (Tk >= 1) {
        const double msq = a2 / (double)Tk;
        mean = a1 / (double)Tk;
        var = msq - mean * mean;
        cancel = msq > 0.0 && !(var >= 1e-8 * msq); // over half of float64's digits cancelled: |mean| > 10^4 sigma
    }
    if (__any_sync(0xffffffffu, cancel)) { // exact two-pass variance about the mean (reading R31)
        double c1 = 0.0, c2 = 0.0;
        stats_whole(U, rbase + (P.lo - P.ring_lo) * (NCHAN * 32), (int)Tk, true, mean, c1, c2);
        if (cancel) var = c2 / (double)Tk;
    }
    if (live) {
        P.s1[o] = a1;
        P.s2[o] = a2;
    }
    if (Tk >= 1) {
        if (!(var > 0.0) && var == var) var = 0.0; // (a NaN stays a NaN: non-finite data in the ring)
        const double sigma = sqrt(var);
        m = (float)mean;
        dl = (float)(mean - (double)m);
        rs = sigma > 0.0 ? (float)(1.0 / sigma) : (sigma == sigma ? 0.f : __int_as_float(0x7fc00000));
        sg = (float)sigma;
    }
    if (!live) return;
    P.mu[o] = m;
    P.dlt[o] = dl;
    P.rsig[o] = rs;
    if (P.sig_out) P.sig_out[o] = sg;
}

} // namespace sk

extern "C" __global__ void __launch_bounds__(256) k_stream_stats(const StatsParams P)
{
    const int lane = threadIdx.x & 31;
    const int u = blockIdx.y * (blockDim.x >> 5) + (threadIdx.x >> 5); // warp = trial; the warps of a CTA share the raw rows in L1
    if (u >= NU) return;
    int pix = blockIdx.x * 32 + lane;
    const bool live = pix < NPIX;
    if (!live) pix = NPIX - 1;
    sk::stats_trial(P, u, lane, pix, live);
}
#endif

#endif
