// k_stream: the hot kernel of nsfrb_stream_push (steps a1..a6 of DESIGN.md) for sm_100a.
//
// This file is compiled AT PLAN TIME (NVRTC, sm_100a) behind a generated prologue that fixes the
// plan's constants -- NPIX, NCHAN, the delay table, the width list, the tile shape -- so every
// dedispersion shift is an immediate and every register array is statically indexed (PAPER.md:L75:
// "shift indices for each frequency channel [are] pre-computed and loaded onto the GPU to minimize
// latencies"; here they are compiled into the instruction stream).  `build()` also compiles it
// ahead of time with the BASELINE config-2 prologue as a build check.
//
// Prologue (see nsfrb_jit.cu: make_stream_prologue):
//   NPIX NCHAN NU KK GPC SEG TT NW CMAX NSUPER MINB     integers
//   E_TAB[NU][NCHAN]   reverse-frame delays  e[u][c] = dmax_u - d[u][c]   (unique trials, DM ascending)
//   DMAX_TAB[NU]       dmax_u                 K_OF_U[NU]  lowest original dm index of the trial
//   W_TAB[NW]          widths, ascending      J_OF_W[NW]  original width index
//
// Reverse frame.  The ring holds raw samples rho in [0, len); s = len-1-rho counts back from the
// newest one.  Series u has T_u = len - dmax_u samples; its r-th sample from the end (r = 1..T_u) is
//     D_u(r) = sum_c R[c][s = (r-1) + e[u][c]]
// i.e. a dedispersion in reversed time with delays e, aligned over u at the ring's newest edge.
// With Q_u(r) = sum_{r'<=r} (D_u(r') - mu0_u) (suffix sums of the series), the boxcar of width w whose
// window excludes the newest i samples is B(i, w) = Q(i+w) - Q(i); rule S5 (only windows whose last
// raw sample arrived in this push) keeps exactly i in [0, chunk_nt) for every trial.  One backward
// march therefore needs, per (pixel, trial): Q (register), Q at the C ends (shared memory, Qe) and
// the running max per width (shared memory, M) -- no prefix history, no P ring.
//
// Mapping.  Lane = pixel (the ring is pixel-contiguous: every load is one coalesced 128-byte row
// segment).  Thread = 1 pixel x KK consecutive trials x 1 of SEG time segments.  A tile is TT steps:
// the thread holds the raw window of every channel in registers (TT new rows + a carried halo of
// span_c = max_kk e - min_kk e rows), forms D for its first trial as the plain channel sum and every
// next trial differentially (a2), then x = D - mu0, Q += x, S2 += x^2 (a1, a3, a4).  Tiles that touch
// a width's start range also evaluate its cells (a5).  Segments are cut between start ranges, so a
// width belongs to one segment and its maxima are relative to that segment's offset, added at the end.
// End of march: delta = S1/T, var = S2/T - delta^2, S = (M + Off - w delta)/(sigma sqrt(w)), reduced over
// widths, trials and DM groups of the CTA (a6).  Raw rows for tile n+1 are requested before tile n
// is computed (register double buffer).
#ifndef NSFRB_STREAM_KERNEL_CUH
#define NSFRB_STREAM_KERNEL_CUH

struct SPartial { // per (pixel, slice): slice = pass * NSUPER + supergroup
    float snr;
    int k, j, t; // original dm index, original width index, window start relative to ring sample 0
};

struct StreamParams {
    const float *ring; // [rows][NCHAN][NPIX], baseline removed, every sample stored at slot and slot+L
    float *mu0;        // [NU][NPIX] provisional means (the previous push's exact means); updated
    SPartial *partials;
    int top_row; // row of the newest sample
    int len;     // valid raw samples in the ring
    int i0, C;   // this pass evaluates ends i in [i0, i0+C)
    int nslice, slice0;
    int rfast;          // steps r <= rfast are valid for every trial (len - dmax_all, >= 0)
    int bound[9];       // segment q < SEG marches steps (bound[q], bound[q+1]], multiples of TT (SEG <= 8)
};

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
    static __host__ __device__ constexpr int e(int kk, int c) { return E_TAB[u(kk)][c]; }
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
constexpr int kTrialsPerCta = GPC * KK;

// shared memory: Qe[kTrialsPerCta][CMAX][32], M[kTrialsPerCta][NW][32], A (uint8) same shape as M,
// S1[kTrialsPerCta][SEG][32], S2 same, then the cross-group reduction scratch
constexpr int kQeFloats = kTrialsPerCta * CMAX * 32;
constexpr int kMFloats = kTrialsPerCta * NW * 32;
constexpr int kSegFloats = kTrialsPerCta * SEG * 32;
constexpr int kRedFloats = GPC * 32 * 4;
constexpr int kSmemBytes = (kQeFloats + kMFloats + 2 * kSegFloats + kRedFloats) * 4 + kMFloats /*A bytes*/;

__device__ __forceinline__ float ldrow(const float *p) { return __ldg(p); }

template <int G> struct Worker {
    using T = GT<G>;
    const float *rp; // &ring[top_row][0][pixel]
    float *qe;       // &Qe[gl*KK][0][lane]
    float *ms;       // &M [gl*KK][0][lane]
    unsigned char *as; // &A[gl*KK][0][lane]
    int lane, i0, C, len;
    float carry[T::CARRY];
    float mu[KK], Q[KK], S2[KK];
    int ja, jb; // widths [ja, jb) can have cells in the current tile

    // element m of channel c's window at tile base rb lives at reverse raw index s = rb + m + emin(c)
    template <int C_, int M_> __device__ __forceinline__ const float *addr(int rb) const
    {
        return rp + ((long long)C_ - (long long)(M_ + T::emin(C_)) * NCHAN) * NPIX - (long long)rb * NCHAN * NPIX;
    }
    __device__ __forceinline__ void load_new(float (&buf)[NCHAN * TT], int rb) const
    {
        const float *b = rp - (long long)rb * NCHAN * NPIX;
        sfor<0, NCHAN>([&](auto c) {
            sfor<0, TT>([&](auto tt) {
                constexpr long long off = ((long long)V(c) - (long long)(T::span(V(c)) + V(tt) + T::emin(V(c))) * NCHAN) * NPIX;
                buf[V(c) * TT + V(tt)] = ldrow(b + off);
            });
        });
    }
    __device__ __forceinline__ void load_carry(int rb)
    {
        const float *b = rp - (long long)rb * NCHAN * NPIX;
        sfor<0, NCHAN>([&](auto c) {
            sfor<0, T::span(V(c))>([&](auto m) {
                constexpr long long off = ((long long)V(c) - (long long)(V(m) + T::emin(V(c))) * NCHAN) * NPIX;
                carry[T::coff(V(c)) + V(m)] = ldrow(b + off);
            });
        });
    }

    // one tile: steps rb+1 .. rb+TT.  cur = the TT new rows of every channel; nxt receives the next tile's.
    template <bool CELLS, bool MASKED>
    __device__ __forceinline__ void tile(float (&cur)[NCHAN * TT], float (&nxt)[NCHAN * TT], int rb, bool prefetch)
    {
        if (prefetch) load_new(nxt, rb + TT);
        auto Wn = [&](auto c, auto m) -> float {
            if constexpr (V(m) < T::span(V(c))) return carry[T::coff(V(c)) + V(m)];
            else return cur[V(c) * TT + (V(m) - T::span(V(c)))];
        };
        float D[TT];
        float Qs[KK][TT];
        sfor<0, KK>([&](auto kk) {
            if constexpr (V(kk) == 0) {
                sfor<0, TT>([&](auto tt) {
                    float a0 = 0.f, a1 = 0.f;
                    sfor<0, NCHAN>([&](auto c) {
                        const float v = Wn(c, IC<V(tt) + T::o(0, V(c))>{});
                        if constexpr ((V(c) & 1) == 0) a0 += v; else a1 += v;
                    });
                    D[V(tt)] = a0 + a1;
                });
            } else {
                sfor<0, TT>([&](auto tt) {
                    float a = 0.f;
                    sfor<0, NCHAN>([&](auto c) {
                        if constexpr (T::o(V(kk), V(c)) != T::o(V(kk) - 1, V(c)))
                            a += Wn(c, IC<V(tt) + T::o(V(kk), V(c))>{}) - Wn(c, IC<V(tt) + T::o(V(kk) - 1, V(c))>{});
                    });
                    D[V(tt)] += a;
                });
            }
            // a1, a3, a4: centred sample, suffix sum, sum of squares
            sfor<0, TT>([&](auto tt) {
                float x = D[V(tt)] - mu[V(kk)];
                if constexpr (MASKED) x = ((rb + 1 + V(tt)) <= len - DMAX_TAB[T::u(V(kk))]) ? x : 0.f;
                Q[V(kk)] += x;
                S2[V(kk)] = fmaf(x, x, S2[V(kk)]);
                Qs[V(kk)][V(tt)] = Q[V(kk)];
            });
            if constexpr (CELLS) {
                if (G * KK + V(kk) < NU) {
                    // Q at the ends of this pass: Qe[ii] = Q(i0 + ii)
                    sfor<0, TT>([&](auto tt) {
                        const int ii = rb + 1 + V(tt) - i0;
                        if (ii >= 0 && ii < C) qe[(V(kk) * CMAX + ii) * 32] = Qs[V(kk)][V(tt)];
                    });
                }
            }
        });
        if constexpr (CELLS) {
            // a5: widths whose start range [w+i0, w+i0+C-1] meets this tile
            while (ja < NW && W_TAB[ja] + i0 + C - 1 < rb + 1) ++ja;
            while (jb < NW && W_TAB[jb] + i0 <= rb + TT) ++jb;
            for (int j = ja; j < jb; ++j) {
                const int ib = rb + 1 - W_TAB[j] - i0; // end index (relative to i0) of step rb+1
                sfor<0, KK>([&](auto kk) {
                    if (G * KK + V(kk) < NU) {
                        float m = ms[(V(kk) * NW + j) * 32];
                        int a = as[(V(kk) * NW + j) * 32];
                        sfor<0, TT>([&](auto tt) {
                            const int ii = ib + V(tt);
                            bool in = (ii >= 0) && (ii < C);
                            if constexpr (MASKED) in = in && ((rb + 1 + V(tt)) <= len - DMAX_TAB[T::u(V(kk))]);
                            if (in) {
                                const float v = Qs[V(kk)][V(tt)] - qe[(V(kk) * CMAX + ii) * 32];
                                if (v >= m) { m = v; a = ii; } // later step = earlier start: ties go to the smaller t
                            }
                        });
                        ms[(V(kk) * NW + j) * 32] = m;
                        as[(V(kk) * NW + j) * 32] = (unsigned char)a;
                    }
                });
            }
        }
        // carry the halo: next tile's element m is this tile's element m + TT
        float nc[T::CARRY];
        sfor<0, NCHAN>([&](auto c) {
            sfor<0, T::span(V(c))>([&](auto m) { nc[T::coff(V(c)) + V(m)] = Wn(c, IC<V(m) + TT>{}); });
        });
        sfor<0, T::CARRY>([&](auto i) { carry[V(i)] = nc[V(i)]; });
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

template <int G> __device__ __forceinline__ void run_group(const StreamParams &P, float *smem, int gl, int seg, int lane, int pix, bool live)
{
    using T = GT<G>;
    float *Qe = smem;
    float *Ms = Qe + kQeFloats;
    float *S1s = Ms + kMFloats;
    float *S2s = S1s + kSegFloats;
    float *red = S2s + kSegFloats;
    unsigned char *As = reinterpret_cast<unsigned char *>(red + kRedFloats);

    Worker<G> w;
    w.lane = lane; w.i0 = P.i0; w.C = P.C; w.len = P.len;
    w.rp = P.ring + ((long long)P.top_row * NCHAN) * NPIX + pix;
    w.qe = Qe + (gl * KK) * CMAX * 32 + lane;
    w.ms = Ms + (gl * KK) * NW * 32 + lane;
    w.as = As + (gl * KK) * NW * 32 + lane;
    w.ja = 0; w.jb = 0;
    sfor<0, KK>([&](auto kk) {
        w.mu[V(kk)] = P.mu0[(long long)T::u(V(kk)) * NPIX + pix];
        w.Q[V(kk)] = 0.f;
        w.S2[V(kk)] = 0.f;
    });
    // this thread initialises the M/A slots of its trials for the widths of its segment ... all segments
    // share the slots, so segment 0 initialises everything before the first barrier
    if (seg == 0) {
        for (int j = 0; j < NW; ++j)
            sfor<0, KK>([&](auto kk) {
                w.ms[(V(kk) * NW + j) * 32] = -kInf;
                w.as[(V(kk) * NW + j) * 32] = 0;
            });
        if (P.i0 == 0) sfor<0, KK>([&](auto kk) { w.qe[(V(kk) * CMAX) * 32] = 0.f; });
    }

    const int r_begin = P.bound[seg], r_end = P.bound[seg + 1];
    const int qe_end = P.i0 + P.C; // steps < qe_end store Qe (they all lie in segment 0)
    bool synced = false;
    if (r_begin < r_end) {
        float bufA[NCHAN * TT], bufB[NCHAN * TT];
        w.load_carry(r_begin);
        w.load_new(bufA, r_begin);
        int rb = r_begin;
        bool flip = false;
        while (rb < r_end) {
            const bool pf = rb + TT < r_end;
            const bool masked = rb + TT > P.rfast;
            // does the tile store ends or touch a start range?
            bool cells = rb < qe_end;
            if (!cells) {
                int ja = w.ja;
                while (ja < NW && W_TAB[ja] + P.i0 + P.C - 1 < rb + 1) ++ja;
                w.ja = ja;
                cells = ja < NW && W_TAB[ja] + P.i0 <= rb + TT;
            }
            if (cells && seg != 0 && !synced) { // Qe is complete once segment 0 has passed qe_end
                bar_named(1, kThreads);
                synced = true;
            }
            if (!flip) {
                if (masked) w.template tile<true, true>(bufA, bufB, rb, pf);
                else if (cells) w.template tile<true, false>(bufA, bufB, rb, pf);
                else w.template tile<false, false>(bufA, bufB, rb, pf);
            } else {
                if (masked) w.template tile<true, true>(bufB, bufA, rb, pf);
                else if (cells) w.template tile<true, false>(bufB, bufA, rb, pf);
                else w.template tile<false, false>(bufB, bufA, rb, pf);
            }
            flip = !flip;
            rb += TT;
            if (seg == 0 && !synced && rb >= qe_end) {
                bar_named(1, kThreads);
                synced = true;
            }
        }
    }
    if (!synced) bar_named(1, kThreads);

    // segment totals
    sfor<0, KK>([&](auto kk) {
        S1s[((gl * KK + V(kk)) * SEG + seg) * 32 + lane] = w.Q[V(kk)];
        S2s[((gl * KK + V(kk)) * SEG + seg) * 32 + lane] = w.S2[V(kk)];
    });
    bar_named(2, kThreads);

    // a6: exact mean/variance, normalise, reduce over widths and trials (segment-0 threads)
    float bs = -kInf;
    int bk = -1, bj = -1, bt = -1;
    if (seg == 0) {
        sfor<0, KK>([&](auto kk) {
            constexpr int u = G * KK + V(kk);
            if constexpr (u < NU) {
                const int Tk = P.len - DMAX_TAB[u];
                if (Tk >= 1) {
                    float off[SEG];
                    float s1 = 0.f, s2 = 0.f;
                    sfor<0, SEG>([&](auto q) {
                        off[V(q)] = s1;
                        s1 += S1s[((gl * KK + V(kk)) * SEG + V(q)) * 32 + lane];
                        s2 += S2s[((gl * KK + V(kk)) * SEG + V(q)) * 32 + lane];
                    });
                    const float invT = 1.f / (float)Tk;
                    const float delta = s1 * invT;
                    const float var = fmaxf(fmaf(-delta, delta, s2 * invT), 0.f);
                    const float sigma = sqrtf(var);
                    if (P.slice0 == 0 && live) P.mu0[(long long)u * NPIX + pix] = w.mu[V(kk)] + delta;
                    for (int j = 0; j < NW; ++j) {
                        const float m = w.ms[(V(kk) * NW + j) * 32];
                        if (m > -kInf) {
                            const int wj = W_TAB[j];
                            const int rj = wj + P.i0; // first start step of the width: fixes its segment
                            float o = 0.f;
                            sfor<1, SEG>([&](auto q) { if (rj > P.bound[V(q)]) o = off[V(q)]; });
                            const float fw = (float)wj;
                            const float B = fmaf(-fw, delta, m + o);
                            const float S = sigma > 0.f ? B / (sigma * sqrtf(fw)) : 0.f;
                            const int ii = P.i0 + (int)w.as[(V(kk) * NW + j) * 32];
                            const int t = Tk - ii - wj;
                            if (better(S, K_OF_U[u], J_OF_W[j], t, bs, bk, bj, bt)) { bs = S; bk = K_OF_U[u]; bj = J_OF_W[j]; bt = t; }
                        }
                    }
                }
            }
        });
        red[(gl * 32 + lane) * 4 + 0] = bs;
        reinterpret_cast<int *>(red)[(gl * 32 + lane) * 4 + 1] = bk;
        reinterpret_cast<int *>(red)[(gl * 32 + lane) * 4 + 2] = bj;
        reinterpret_cast<int *>(red)[(gl * 32 + lane) * 4 + 3] = bt;
    }
    bar_named(3, kThreads);
    if (seg == 0 && gl == 0 && live) {
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

template <int G0, int N> __device__ __forceinline__ void dispatch(int g, const StreamParams &P, float *smem, int gl, int seg, int lane, int pix, bool live)
{
    if constexpr (N == 1) {
        run_group<G0>(P, smem, gl, seg, lane, pix, live);
    } else {
        if (g < G0 + N / 2) dispatch<G0, N / 2>(g, P, smem, gl, seg, lane, pix, live);
        else dispatch<G0 + N / 2, N - N / 2>(g, P, smem, gl, seg, lane, pix, live);
    }
}

} // namespace sk

extern "C" __global__ void __launch_bounds__(sk::kThreads, MINB) k_stream(const StreamParams P)
{
    extern __shared__ __align__(16) float smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int gl = warp / SEG, seg = warp - gl * SEG;
    // pixel blocks past NPIX clamp to the last pixel (loads stay in bounds; the store is skipped)
    int pix = blockIdx.x * 32 + lane;
    const bool live = pix < NPIX;
    if (!live) pix = NPIX - 1;
    const int g = blockIdx.y * GPC + gl; // DM group of this warp; NSUPER*GPC groups exist (padded)
    sk::dispatch<0, NSUPER * GPC>(g, P, smem, gl, seg, lane, pix, live);
}

#endif
