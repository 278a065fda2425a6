// NEXT 4 of SURVEY.md 8(f): the imaging step that feeds the search for sm_100a.
//
//   nsfrb_imager_create   host, float64: baseline selection (20 m < b < 485 m), nearest UV cell of every (channel, baseline),
//                         Briggs weights (R = -2), normalisation -- everything that does not depend on the data
//   nsfrb_imager_image    one launch of k_image per call: visibilities [nt][nchan][nbase][2 pol] complex64 -> images [nt][n][n]
//
// k_image.  The paper grids each channel, applies ifftshift / ifft2 / ifftshift and sums the 8 channel images (L61, L67).
// The transform is linear and the grid Hermitian, so one CTA = one time sample x 32 image columns does it as a separable
// inverse DFT over the SPARSE visibility list, all channels at once, in the half plane fv >= 0:
//   phase 1  R[r][x] = sum over the entries of row r = |fv| of  a_i Vc_i tw[fu_i (x - x0) mod n]     (Vc = V for fv >= 0, conj V and
//            -fu for fv < 0; V = the two polarisations summed; a_i = Briggs weight / sum of the channel's weights)
//            warps take rows, lanes take columns; 32 visibilities at a time are loaded coalesced and broadcast by shuffles;
//            the twiddle is a shared-memory table
//   phase 2  I[y][x] = 2 sum_r Re(R[r][x] tw[r (y - x0) mod n])                                    (the other half plane is the conjugate)
// with x0 = n - n / 2 the pixel the paper's final ifftshift puts the phase centre on.  Same result as the oracle's route up
// to float32 rounding; shares no code with oracle/imaging.py.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "nsfrb_internal.h"

struct nsfrb_imager {
    int n = 0, nchan = 0, nbase = 0, device = 0;
    std::vector<int32_t> cells;   // [nchan][nbase][2] (fu, fv); meaningful where weight > 0
    std::vector<double> weights;  // [nchan][nbase] Briggs weight, 0 = not gridded
    int nentries = 0;
    // device
    int2 *d_entry = nullptr;      // [nentries] (visibility index | conj << 31, fu), sorted by row
    float *d_coeff = nullptr;     // [nentries]
    int *d_row = nullptr;         // [nunit][3] work units (row |fv|, first entry, one past the last): <= 256 entries of one row each
    int nunit = 0;
    float2 *d_tw = nullptr;       // [n] exp(2 pi i k / n)
};

namespace nsfrb {
namespace {

constexpr int kImgThreads = 512;

struct ImageParams {
    const float4 *vis;  // [nt][nchan*nbase] (re0, im0, re1, im1)
    const int2 *entry;
    const float *coeff;
    const int *unit;    // [nunit][3]
    const float2 *tw;
    float *out;         // [nt][n][n]
    int n, nvis, nrow, nunit;  // nvis = nchan*nbase; nrow = n/2 + 1
};

__global__ void __launch_bounds__(kImgThreads) k_image(const ImageParams P)
{
    extern __shared__ __align__(16) float2 sm[]; // tw[n] | R[nrow][32]
    float2 *tw = sm;
    float2 *R = sm + P.n;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = kImgThreads / 32;
    const int t = blockIdx.y, x = blockIdx.x * 32 + lane;
    const int n = P.n, x0 = n - n / 2;
    __shared__ int next_unit;
    if (threadIdx.x == 0) next_unit = 0;
    for (int i = threadIdx.x; i < n; i += kImgThreads) tw[i] = P.tw[i];
    for (int i = threadIdx.x; i < P.nrow * 32; i += kImgThreads) R[i] = make_float2(0.f, 0.f);
    __syncthreads();
    const int dx = x - x0;
    const float4 *vt = P.vis + (size_t)t * P.nvis;
    // ---- phase 1: rows of the half plane, in work units of <= 256 entries of one row (an east-west array puts most of its
    // visibilities into the rows next to fv = 0: a row per warp would leave one warp with half the work).  Warps take units
    // from a shared counter; per 32 entries every lane loads one (coalesced, independent loads) and forms its weighted,
    // polarisation-summed, possibly conjugated visibility; the 32 are then broadcast one by one; a unit's partial sums are
    // added to the row with shared-memory atomics (the order of those additions is the only run-to-run freedom: ~1e-7).
    const unsigned M = 0xffffffffu / (unsigned)n + 1u; // ceil(2^32 / n): umulhi(p, M) = floor(p / n), or that + 1 for large p
    const int bias = n * (n + 1);                       // > |fu dx|: makes the product non-negative, and is 0 mod n
    for (;;) {
        int ui = 0;
        if (lane == 0) ui = atomicAdd(&next_unit, 1);
        ui = __shfl_sync(0xffffffffu, ui, 0);
        if (ui >= P.nunit) break;
        float re = 0.f, im = 0.f;
        const int r = P.unit[3 * ui], e0 = P.unit[3 * ui + 1], e1 = P.unit[3 * ui + 2];
        for (int eb = e0; eb < e1; eb += 32) {
            const int e = eb + lane;
            float vr = 0.f, vi = 0.f;
            int fu = 0;
            if (e < e1) {
                const int2 en = __ldg(P.entry + e);
                const float a = __ldg(P.coeff + e);
                const float4 v = __ldg(vt + (en.x & 0x7fffffff));
                vr = a * (v.x + v.z);                          // pols summed (L55)
                vi = (en.x < 0 ? -a : a) * (v.y + v.w);        // conjugate for fv < 0
                fu = en.y;
            }
            const int cnt = e1 - eb < 32 ? e1 - eb : 32;
            for (int j = 0; j < cnt; ++j) {
                const float br = __shfl_sync(0xffffffffu, vr, j), bi = __shfl_sync(0xffffffffu, vi, j);
                const unsigned p = (unsigned)(__shfl_sync(0xffffffffu, fu, j) * dx + bias);
                int k = (int)(p - (unsigned)n * __umulhi(p, M)); // the quotient may be one too large (never too small)
                k = k < 0 ? k + n : k;
                const float2 w = tw[k];
                re = fmaf(br, w.x, fmaf(-bi, w.y, re));
                im = fmaf(br, w.y, fmaf(bi, w.x, im));
            }
        }
        atomicAdd(&R[r * 32 + lane].x, re);
        atomicAdd(&R[r * 32 + lane].y, im);
    }
    __syncthreads();
    // ---- phase 2: columns
    if (x >= n) return;
    for (int y = warp; y < n; y += nwarp) {
        int dy = y - x0;
        dy = dy < 0 ? dy + n : dy; // step of the twiddle index per row
        int k = 0;
        float a0 = 0.f, a1 = 0.f;
        for (int r = 0; r < P.nrow; ++r) {
            const float2 v = R[r * 32 + lane], w = tw[k];
            if (r & 1) a1 = fmaf(v.x, w.x, fmaf(-v.y, w.y, a1));
            else a0 = fmaf(v.x, w.x, fmaf(-v.y, w.y, a0));
            k += dy;
            k = k >= n ? k - n : k;
        }
        P.out[((size_t)t * n + y) * n + x] = 2.f * (a0 + a1);
    }
}

} // namespace
} // namespace nsfrb

#pragma GCC visibility push(default)
extern "C" {

int nsfrb_imager_create(nsfrb_imager **out, int n, double pixel_rad, const double *uv_m, int nbase, const double *freqs_GHz,
                        int nchan, double bmin_m, double bmax_m, double robust)
{
    using nsfrb::api_fail;
    if (!out) return api_fail(NSFRB_EINVAL, "out is null");
    *out = nullptr;
    if (!uv_m || !freqs_GHz) return api_fail(NSFRB_EINVAL, "null input list");
    if (n < 2 || n > 2048 || nbase < 1 || nchan < 1) return api_fail(NSFRB_EINVAL, "size out of range (2 <= n <= 2048)");
    if (!(pixel_rad > 0.0) || !std::isfinite(pixel_rad) || !(bmax_m > bmin_m) || !std::isfinite(robust))
        return api_fail(NSFRB_EINVAL, "pixel_rad must be > 0, bmax_m > bmin_m, robust finite");
    if ((long long)nchan * nbase > 0x3fffffffLL) return api_fail(NSFRB_EINVAL, "too many visibilities");
    for (int c = 0; c < nchan; ++c)
        if (!(freqs_GHz[c] > 0.0) || !std::isfinite(freqs_GHz[c])) return api_fail(NSFRB_EINVAL, "freqs_GHz must be finite and > 0");
    nsfrb_imager *im = new (std::nothrow) nsfrb_imager();
    if (!im) return api_fail(NSFRB_ENOMEM, "host allocation failed");
    im->n = n; im->nchan = nchan; im->nbase = nbase;
    im->cells.assign((size_t)nchan * nbase * 2, 0);
    im->weights.assign((size_t)nchan * nbase, 0.0);
    const int c0 = n / 2;
    std::vector<double> W((size_t)n * n);
    struct Entry { int row, idx, fu; bool conj; double a; };
    std::vector<Entry> entries;
    for (int ch = 0; ch < nchan; ++ch) {
        // I1: metres -> cells: u_lambda = u_m f / c, cell size 1 / (n pixel_rad)
        const double scale = (freqs_GHz[ch] * 1.0e9 / 299792458.0) * ((double)n * pixel_rad);
        std::fill(W.begin(), W.end(), 0.0);
        std::vector<char> inside(nbase, 0);
        double nvis = 0.0;
        for (int b = 0; b < nbase; ++b) {
            const double u = uv_m[2 * b], v = uv_m[2 * b + 1];
            const double len = std::sqrt(u * u + v * v);
            if (!(len > bmin_m && len < bmax_m)) continue;                     // L55: b_min < b < b_max
            const long long fu = (long long)std::floor(u * scale + 0.5), fv = (long long)std::floor(v * scale + 0.5);
            im->cells[((size_t)ch * nbase + b) * 2] = (int32_t)fu;
            im->cells[((size_t)ch * nbase + b) * 2 + 1] = (int32_t)fv;
            if (c0 + fu < 0 || c0 + fu >= n || c0 - fu < 0 || c0 - fu >= n || c0 + fv < 0 || c0 + fv >= n || c0 - fv < 0 || c0 - fv >= n)
                continue;                                                       // off the grid
            inside[b] = 1;
            W[(size_t)(c0 + fv) * n + (c0 + fu)] += 1.0;                        // the visibility and its Hermitian copy
            W[(size_t)(c0 - fv) * n + (c0 - fu)] += 1.0;
            nvis += 2.0;
        }
        if (nvis == 0.0) continue;
        double sw2 = 0.0;
        for (double w : W) sw2 += w * w;
        const double f2 = std::pow(5.0 * std::pow(10.0, -robust), 2.0) / (sw2 / nvis); // I3: Briggs 1995
        double wsum = 0.0;
        for (int b = 0; b < nbase; ++b)
            if (inside[b]) {
                const int fu = im->cells[((size_t)ch * nbase + b) * 2], fv = im->cells[((size_t)ch * nbase + b) * 2 + 1];
                const double w = 1.0 / (1.0 + W[(size_t)(c0 + fv) * n + (c0 + fu)] * f2);
                im->weights[(size_t)ch * nbase + b] = w;
                wsum += 2.0 * w;
            }
        for (int b = 0; b < nbase; ++b) {
            const double w = im->weights[(size_t)ch * nbase + b];
            if (w == 0.0) continue;
            const int fu = im->cells[((size_t)ch * nbase + b) * 2], fv = im->cells[((size_t)ch * nbase + b) * 2 + 1];
            // I4: unit point-source response; the n^2 of the normalisation cancels ifft2's 1 / n^2
            entries.push_back({fv >= 0 ? fv : -fv, ch * nbase + b, fv >= 0 ? fu : -fu, fv < 0, w / wsum});
        }
    }
    std::stable_sort(entries.begin(), entries.end(), [](const Entry &a, const Entry &b) { return a.row < b.row; });
    std::vector<int2> h_entry(std::max<size_t>(entries.size(), 1));
    std::vector<float> h_coeff(std::max<size_t>(entries.size(), 1), 0.f);
    std::vector<int> h_row; // work units (row, e0, e1), heaviest rows first in the list order of the sort (row 0 upwards)
    for (size_t i = 0; i < entries.size(); ++i) {
        h_entry[i] = make_int2(entries[i].idx | (entries[i].conj ? (int)0x80000000u : 0), entries[i].fu);
        h_coeff[i] = (float)entries[i].a;
    }
    for (size_t i = 0; i < entries.size();) {
        size_t j = i;
        while (j < entries.size() && entries[j].row == entries[i].row && j - i < 256) ++j;
        h_row.push_back(entries[i].row); h_row.push_back((int)i); h_row.push_back((int)j);
        i = j;
    }
    im->nunit = (int)(h_row.size() / 3);
    if (h_row.empty()) h_row.assign(3, 0);
    std::vector<float2> h_tw(n);
    for (int k = 0; k < n; ++k) h_tw[k] = make_float2((float)std::cos(2.0 * M_PI * k / n), (float)std::sin(2.0 * M_PI * k / n));
    im->nentries = (int)entries.size();
    cudaError_t e = cudaGetDevice(&im->device);
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&im->d_entry), h_entry.size() * sizeof(int2));
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&im->d_coeff), h_coeff.size() * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&im->d_row), h_row.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&im->d_tw), h_tw.size() * sizeof(float2));
    if (e == cudaSuccess) e = cudaMemcpy(im->d_entry, h_entry.data(), h_entry.size() * sizeof(int2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(im->d_coeff, h_coeff.data(), h_coeff.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(im->d_row, h_row.data(), h_row.size() * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(im->d_tw, h_tw.data(), h_tw.size() * sizeof(float2), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        const std::string msg = std::string("imager device setup: ") + cudaGetErrorString(e);
        cudaGetLastError();
        nsfrb_imager_destroy(im);
        return api_fail(e == cudaErrorMemoryAllocation ? NSFRB_ENOMEM : NSFRB_ECUDA, msg);
    }
    *out = im;
    return NSFRB_OK;
}

int nsfrb_imager_image(nsfrb_imager *im, const float *vis, int nt, float *out, void *stream)
{
    using nsfrb::api_fail;
    if (!im) return api_fail(NSFRB_EINVAL, "imager is null");
    if (!vis || !out) return api_fail(NSFRB_EINVAL, "null pointer");
    if ((reinterpret_cast<uintptr_t>(vis) & 15u) != 0) return api_fail(NSFRB_EINVAL, "vis is not 16-byte aligned");
    if (nt < 1 || nt > 65535) return api_fail(NSFRB_EINVAL, "nt out of range (1..65535)");
    nsfrb::ImageParams P;
    P.vis = reinterpret_cast<const float4 *>(vis); P.entry = im->d_entry; P.coeff = im->d_coeff; P.unit = im->d_row; P.tw = im->d_tw;
    P.out = out; P.n = im->n; P.nvis = im->nchan * im->nbase; P.nrow = im->n / 2 + 1; P.nunit = im->nunit;
    const size_t smem = ((size_t)im->n + (size_t)P.nrow * 32) * sizeof(float2);
    static size_t granted[64] = {0};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess && dev >= 0 && dev < 64 && smem > granted[dev] && smem > 48 * 1024) {
        e = cudaFuncSetAttribute(nsfrb::k_image, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) granted[dev] = smem;
    }
    if (e == cudaSuccess) {
        nsfrb::k_image<<<dim3((im->n + 31) / 32, nt), nsfrb::kImgThreads, smem, static_cast<cudaStream_t>(stream)>>>(P);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        const std::string msg = std::string("k_image launch: ") + cudaGetErrorString(e);
        cudaGetLastError();
        return api_fail(NSFRB_ECUDA, msg);
    }
    return NSFRB_OK;
}

int nsfrb_imager_get_table(const nsfrb_imager *im, int32_t *cells, double *weights)
{
    if (!im || !cells || !weights) return nsfrb::api_fail(NSFRB_EINVAL, "null argument");
    std::memcpy(cells, im->cells.data(), im->cells.size() * sizeof(int32_t));
    std::memcpy(weights, im->weights.data(), im->weights.size() * sizeof(double));
    return NSFRB_OK;
}

int nsfrb_imager_destroy(nsfrb_imager *im)
{
    if (!im) return NSFRB_OK;
    cudaFree(im->d_entry); cudaFree(im->d_coeff); cudaFree(im->d_row); cudaFree(im->d_tw);
    cudaGetLastError();
    delete im;
    return NSFRB_OK;
}

} // extern "C"
#pragma GCC visibility pop
