// On-chip ceilings of this GPU, measured: the denominators of the "alu" roofline of the offline search
// ("the builder writes two microbenchmarks (FADD/FMNMX chain; conflict-free LDS stream) and uses the
// achieved numbers and the clock actually sustained").  nsfrb_measure_peaks runs one short kernel per instruction mix on
// every SM and reports lane-operations per second (CUDA events) and per clock per SM (clock64 inside the kernel).
//   issue tests    : NACC independent dependency chains per thread, 1024 threads per CTA, 2 CTAs per SM -- every
//                    scheduler always has an eligible warp, so the figure is the pipe's issue rate
//   shared memory  : each lane streams conflict-free words (LDS.32) or 16-byte vectors (LDS.128) out of a 32 KB tile
// None of this is on the search path; bench.py --op peaks prints the table and the offline roofline divides by it.
#include <cuda_runtime.h>

#include "nsfrb_internal.h"

namespace nsfrb {
namespace {

enum PeakTest {
    kFadd = 0,     // FADD chain                         (what a boxcar difference costs)
    kFmnmx,        // FMNMX chain                        (what a running maximum costs)
    kFmnmx3,       // 3-input FMNMX3 chain               (two cells per maximum)
    kFfma,         // FFMA chain                         (sum of squares)
    kPair,         // 2 FADD + 1 FMNMX3                  (the search's cell pair as issued)
    kViaddmnmx,    // VIADDMNMX chain (max(a + b, c) in one integer instruction)
    kIadd3,        // 3-input integer add chain (as compiled: IADD3 / IMAD.IADD)
    kLds32,        // conflict-free LDS.32 stream + FADD
    kLds128,       // conflict-free LDS.128 stream + 4 FADD
    kNumTests
};

constexpr int NACC = 8;

template <int TEST> __global__ void __launch_bounds__(1024, 2) k_peak(int iters, float seed, float *sink, long long *clk)
{
    __shared__ __align__(16) float tile[8192];
    float a[NACC];
    int ia[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) { a[i] = seed * (float)(threadIdx.x + i); ia[i] = (int)threadIdx.x + i; }
    const float b = seed * 1.0001f, c = seed * 0.5f;
    const int ib = (int)(seed * 3.f) + 1;
    if (TEST == kLds32 || TEST == kLds128) {
        for (int i = threadIdx.x; i < 8192; i += blockDim.x) tile[i] = seed * (float)i;
        __syncthreads();
    }
    const long long t0 = clock64();
    if constexpr (TEST == kLds32) {
        const float *p = tile + (threadIdx.x & 31);
        for (int it = 0; it < iters; ++it) {
            const float *q = p + (it & 7) * 1024; // one address per 32 loads: the loads themselves take immediate offsets
#pragma unroll
            for (int k = 0; k < 32; ++k) a[k & (NACC - 1)] += q[((k * 7) & 31) * 32];
        }
    } else if constexpr (TEST == kLds128) {
        const float4 *p = reinterpret_cast<const float4 *>(tile) + (threadIdx.x & 31);
        for (int it = 0; it < iters; ++it) {
            const float4 *q = p + (it & 3) * 512;
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const float4 v = q[((k * 5) & 15) * 32];
                a[0] += v.x; a[1] += v.y; a[2] += v.z; a[3] += v.w;
            }
        }
    } else {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r) {
#pragma unroll
                for (int i = 0; i < NACC; ++i) {
                    if constexpr (TEST == kFadd) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(b));
                    else if constexpr (TEST == kFmnmx) { // max and min alternate: ptxas would fold max(max(a, b), c) into one FMNMX3
                        if (r & 1) asm volatile("min.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(b));
                        else asm volatile("max.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(c));
                    }
                    else if constexpr (TEST == kFmnmx3) asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(b), "f"(c));
                    else if constexpr (TEST == kFfma) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(b), "f"(c));
                    else if constexpr (TEST == kIadd3) ia[i] = ia[i] + ib + ia[(i + 1) & (NACC - 1)]; // a genuine 3-input add
                    else if constexpr (TEST == kViaddmnmx) ia[i] = __viaddmax_s32(ia[i], ib, ia[(i + 1) & (NACC - 1)]);
                }
                if constexpr (TEST == kPair) { // per pair of cells: two differences, one 3-input maximum
#pragma unroll
                    for (int i = 0; i < NACC; i += 2) {
                        float d0, d1;
                        asm volatile("add.rn.f32 %0, %1, %2;" : "=f"(d0) : "f"(a[i]), "f"(b));
                        asm volatile("add.rn.f32 %0, %1, %2;" : "=f"(d1) : "f"(a[i + 1]), "f"(c));
                        asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(d0), "f"(d1));
                        asm volatile("add.rn.f32 %0, %1, %2;" : "=f"(d0) : "f"(a[i + 1]), "f"(b));
                        asm volatile("add.rn.f32 %0, %1, %2;" : "=f"(d1) : "f"(a[i]), "f"(c));
                        asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(a[i + 1]) : "f"(d0), "f"(d1));
                    }
                }
            }
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
    int is = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) { s += a[i]; is += ia[i]; }
    if (s == 12345.678f || is == 0x7ffffff1) sink[0] = s + (float)is; // keeps the chains alive
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}

// warp-level instructions one thread issues per iteration of the timed loop, and lane-operations they stand for
void test_shape(int test, double *instr, double *lane_ops_per_instr)
{
    *lane_ops_per_instr = 32.0;
    switch (test) {
    case kLds32: *instr = 32; break;                   // LDS.32 count (the FADDs ride along)
    case kLds128: *instr = 16; *lane_ops_per_instr = 128.0; break; // words moved per LDS.128
    case kPair: *instr = 8 * (NACC / 2) * 6; break;
    default: *instr = 8 * NACC; break;
    }
}

template <int TEST> cudaError_t run_one(int iters, int grid, float *sink, long long *clk, cudaStream_t st)
{
    k_peak<TEST><<<grid, 1024, 0, st>>>(iters, 1.0f, sink, clk);
    return cudaGetLastError();
}

cudaError_t run_test(int test, int iters, int grid, float *sink, long long *clk, cudaStream_t st)
{
    switch (test) {
    case kFadd: return run_one<kFadd>(iters, grid, sink, clk, st);
    case kFmnmx: return run_one<kFmnmx>(iters, grid, sink, clk, st);
    case kFmnmx3: return run_one<kFmnmx3>(iters, grid, sink, clk, st);
    case kFfma: return run_one<kFfma>(iters, grid, sink, clk, st);
    case kPair: return run_one<kPair>(iters, grid, sink, clk, st);
    case kViaddmnmx: return run_one<kViaddmnmx>(iters, grid, sink, clk, st);
    case kIadd3: return run_one<kIadd3>(iters, grid, sink, clk, st);
    case kLds32: return run_one<kLds32>(iters, grid, sink, clk, st);
    case kLds128: return run_one<kLds128>(iters, grid, sink, clk, st);
    }
    return cudaErrorInvalidValue;
}

} // namespace

int peaks_num_tests() { return kNumTests; }

const char *peaks_name(int t)
{
    static const char *names[kNumTests] = {"fadd", "fmnmx", "fmnmx3", "ffma", "fadd2_fmnmx3_pair", "viaddmnmx", "iadd", "lds32", "lds128"};
    return (t >= 0 && t < kNumTests) ? names[t] : "";
}

// per_s[t]: lane-operations (issue tests) or 4-byte words (shared-memory tests) per second over the whole GPU;
// per_clk_sm[t]: the same per SM clock per SM, from the slowest CTA's clock64 span.
cudaError_t measure_peaks(int iters, double *per_s, double *per_clk_sm, cudaStream_t st)
{
    int dev = 0, nsm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    const int grid = 2 * nsm;
    float *sink = nullptr;
    long long *clk = nullptr;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    e = cudaMalloc(reinterpret_cast<void **>(&sink), 256);
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&clk), grid * sizeof(long long));
    if (e == cudaSuccess) e = cudaEventCreate(&ev0);
    if (e == cudaSuccess) e = cudaEventCreate(&ev1);
    long long *h = new long long[grid];
    for (int t = 0; t < kNumTests && e == cudaSuccess; ++t) {
        for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) { // two warm-ups, the third is kept
            cudaEventRecord(ev0, st);
            e = run_test(t, iters, grid, sink, clk, st);
            cudaEventRecord(ev1, st);
            if (e == cudaSuccess) e = cudaEventSynchronize(ev1);
        }
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, ev0, ev1);
        e = cudaMemcpy(h, clk, grid * sizeof(long long), cudaMemcpyDeviceToHost);
        long long worst = 1;
        for (int i = 0; i < grid; ++i) worst = h[i] > worst ? h[i] : worst;
        double instr, lane;
        test_shape(t, &instr, &lane);
        const double per_cta = instr * lane * (1024.0 / 32.0) * (double)iters;
        per_s[t] = per_cta * grid / ((double)ms * 1e-3);
        per_clk_sm[t] = per_cta * 2.0 / (double)worst; // two CTAs share an SM
    }
    delete[] h;
    cudaFree(sink); cudaFree(clk);
    if (ev0) cudaEventDestroy(ev0);
    if (ev1) cudaEventDestroy(ev1);
    return e;
}

} // namespace nsfrb
