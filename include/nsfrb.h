/*
 * nsfrb.h -- C ABI of the B200-native NSFRB image-plane single-pulse search.
 *
 * The library computes the search stage of the DSA-110 NSFRB pipeline ("cerberus",
 * arxiv 2510.18136 sec. 2.2): per-pixel incoherent dedispersion of a
 * stack of sub-band images over trial DMs, boxcar matched filter over trial widths,
 * S/N normalisation by the per-(pixel, DM) standard deviation, maximum S/N and its time
 * of arrival, and a thresholded candidate list.  Where the paper is silent the readings
 * R1..R23 in DESIGN.md apply.  Every step runs in CUDA kernels for sm_100a; there is no
 * CPU fallback.
 *
 * Notation: npix = nx*ny, pixel p = y*nx + x; cube I[c][t][p] float32, pixel-contiguous,
 * index (c*nt + t)*npix + p.  For DM trial k and channel c the integer delay is
 *     d[k][c] = floor(((4.15e-3*dm[k]) * (f[c]^-2 - f_ref^-2)) / tsamp + 0.5), f_ref = max f
 * (PAPER.md:L83 dispersion constant, L98 integer shift table), T_k = nt - max_c d[k][c].
 *     D_k[t] = sum_c I[c][t+d[k][c]][p]            0 <= t < T_k
 *     S(k,j,t) = sum_{u=t}^{t+w_j-1} (D_k[u]-mu_k) / (sigma_k*sqrt(w_j)),  0 <= t <= T_k-w_j
 * with mu_k, sigma_k the mean and population standard deviation of D_k over all valid t
 * (S = 0 where sigma_k = 0).  Outputs per pixel: snr = max S, argmax = lexicographically
 * smallest (k, j, t) attaining it; candidates = pixels with snr > threshold (strict).
 *
 * Threading: a plan serves one call at a time.  Calls enqueue work on the given stream and
 * return; outputs are valid once the caller has synchronised that stream.  nsfrb_plan_create,
 * nsfrb_plan_prepare, nsfrb_plan_destroy and the *_host variants synchronise the device; so does
 * the FIRST nsfrb_search / nsfrb_stream_push of a plan that was not prepared (it compiles the
 * plan's kernel and allocates its workspaces then); every later call only enqueues.
 * Every call runs on the device that was current at nsfrb_plan_create, whatever device is
 * current in the calling thread, and leaves the caller's current device unchanged.
 * Errors: 0 on success, negative code otherwise; nsfrb_last_error() gives the text.
 */
#ifndef NSFRB_H
#define NSFRB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NSFRB_OK 0
#define NSFRB_EINVAL (-1) /* bad argument (null, non-positive size, bad list, misaligned) */
#define NSFRB_ENOMEM (-2) /* device or host allocation failed / does not fit shared memory */
#define NSFRB_ECUDA (-3)  /* CUDA runtime error; message holds cudaGetErrorString          */
#define NSFRB_ESTATE (-4) /* call not allowed in the plan's state (see nsfrb_search)        */

typedef struct nsfrb_plan nsfrb_plan; /* opaque; owns tables, workspace, ring */

/* One candidate: a pixel whose peak S/N exceeds the threshold ("A nominal
 * 6 sigma S/N threshold is imposed to identify candidates"; L146 one per time series). */
typedef struct {
    int32_t pixel;     /* y*nx + x                                        */
    int32_t dm_idx;    /* index into dm_list (lowest index among duplicates) */
    int32_t width_idx; /* index into width_list                            */
    int32_t t;         /* window start, reference-frequency frame          */
    float snr;
} nsfrb_cand;

/* Sizes and launch facts of a plan, for harnesses (all host values). */
typedef struct {
    int32_t npix, nchan, nt, ndm, nwidth;
    int32_t ndm_unique;        /* distinct delay vectors actually searched           */
    int32_t dmax;              /* largest delay in the table, samples                */
    int32_t wmax;              /* largest width                                      */
    int32_t n_groups;          /* DM groups per pixel (one CTA each)                 */
    int32_t n_width_batches;   /* width batches per pixel (<= 32 widths each)        */
    int32_t series_per_cta;    /* DM trials one CTA holds on chip                    */
    int32_t block_len;         /* dedispersed samples per time block                 */
    int32_t ring_len;          /* prefix-sum history kept per series in shared memory */
    int32_t search_threads;    /* threads per CTA of the search kernel               */
    int64_t search_smem_bytes; /* dynamic shared memory per CTA                      */
    int64_t workspace_bytes;   /* device bytes owned by the plan                     */
    int64_t cells_per_pixel;   /* offline: sum_k sum_j max(0, T_k - w_j + 1), all ndm */
    int64_t shift_adds_per_pixel; /* offline: nchan * sum_k T_k, all ndm            */
} nsfrb_plan_info;

/*
 * Create a plan (DM trials, widths and the shift table are fixed ahead of
 * the search and kept on the GPU).
 *   nx, ny, nchan > 0; nt > 0 is the cube length for nsfrb_search and the ring length L
 *   for nsfrb_stream_push.  freqs_GHz: host [nchan], finite, > 0, any order.  tsamp_s > 0.
 *   dm_list: host [ndm], finite, >= 0.  width_list: host [nwidth], each >= 1, distinct.
 *   Every trial must keep at least one sample: nt > max_c d[k][c] for all k.
 * All host arrays are copied.  Device memory is allocated on the CUDA device current at creation: small tables at creation;
 * at nsfrb_plan_prepare or the first nsfrb_search two pixel-batch workspaces of about 1 GiB each (the search walks the image
 * in batches: no cube-sized buffer) plus ~2 MB of scratch per SM; at nsfrb_plan_prepare or the first nsfrb_stream_push the
 * ring, 2*(nt + guard)*nchan*npix*4 B, the ring of dedispersed samples, 2.25*(nt + guard)*ndm_unique*npix*4 B (left out where
 * it would take more than half of the free device memory: nsfrb_stream_mode), plus a workspace of ~10 B per (pixel, trial,
 * width).  Plans with more than 32 usable
 * widths use a generic kernel with a cube-sized workspace (nchan*nt*npix*4 B).
 */
int nsfrb_plan_create(nsfrb_plan **out, int nx, int ny, int nchan, int nt,
                      const double *freqs_GHz, double tsamp_s,
                      const double *dm_list, int ndm,
                      const int32_t *width_list, int nwidth, float threshold);

/*
 * Optional: do now what the first nsfrb_search / nsfrb_stream_push of a plan would otherwise do lazily -- compile the
 * plan-specialised kernel (NVRTC; seconds to a minute, cached on disk, see NSFRB_JIT_CACHE in DESIGN.md) and allocate
 * the workspaces -- so that those calls only enqueue work.  PAPER.md:L75: the trial grids and shift tables are fixed and
 * "loaded onto the GPU" ahead of the search.
 *   mode NSFRB_PREPARE_SEARCH: offline kernel + two pixel-batch workspaces (about 1 GiB each);
 *        chunk_nt is ignored
 *   mode NSFRB_PREPARE_STREAM: real-time kernel for pushes of chunk_nt samples + the ring and its statistics
 * Synchronises the device (allocation, memset).  Idempotent.  NSFRB_EINVAL for a bad mode or chunk_nt outside [1, nt];
 * NSFRB_ENOMEM / NSFRB_ECUDA as for the calls it prepares (a compile failure carries the NVRTC log).
 */
#define NSFRB_PREPARE_SEARCH 0
#define NSFRB_PREPARE_STREAM 1
int nsfrb_plan_prepare(nsfrb_plan *plan, int mode, int chunk_nt);

/*
 * Offline search of one cube (definition at the top of this file).
 *   cube      device, [nchan][nt][npix] float32, 16-byte aligned, read only
 *   stream    cudaStream_t (NULL = legacy default stream)
 *   snr_map   device, [npix] float32.  -INFINITY where no cell is defined
 *   argmax    device, [3][npix] int32: dm_idx | width_idx | t ; (-1,-1,-1) where no cell
 *   cands     device, [cand_capacity]; may be NULL iff cand_capacity == 0; order arbitrary
 *   ncands    device, 1: total number of candidates found (may exceed cand_capacity, in
 *             which case only cand_capacity of them are stored -- not an error)
 * Returns NSFRB_ESTATE if the plan has received stream pushes (call nsfrb_stream_reset).
 * Non-finite input values give unspecified results.
 */
int nsfrb_search(nsfrb_plan *plan, const float *cube, void *stream,
                 float *snr_map, int32_t *argmax,
                 nsfrb_cand *cands, uint32_t cand_capacity, uint32_t *ncands);

/*
 * Real-time mode (25-sample chunks arrive every 3.35 s and must be
 * searched as they arrive).  Appends chunk [nchan][chunk_nt][npix] (device, 16-byte
 * aligned) to the plan's ring of the last nt samples and searches it:
 *   n_prev -> n = n_prev + chunk_nt samples received; ring = samples [lo, n), lo = max(0, n-nt)
 *   mu_k, sigma_k span every valid sample of the ring; only windows whose LAST raw sample
 *   arrived in this push are evaluated: n_prev <= t + w_j - 1 + dmax_k < n, t >= lo;
 *   reported t is the absolute sample index since the first push (mod 2^31).
 * 1 <= chunk_nt <= nt.  Outputs as nsfrb_search.
 * The sums behind mu_k and sigma_k (sum of D_k and of D_k^2 over the valid samples, float64 per trial and pixel) are
 * plan state carried from push to push: a push adds the samples that enter the valid set and subtracts those that
 * leave it; nsfrb_stream_reset clears them together with the ring.  The memory they take (24 B per trial and pixel) is
 * counted in nsfrb_plan_info's workspace_bytes.  So is the dedispersed sample D_k(t) itself: it is formed once, by the push
 * that brings its last raw sample, and kept in a second ring that later pushes read (nsfrb_stream_mode 2 and 3; DESIGN.md
 * 5.2) -- state with the lifetime of the raw ring, holding nothing the raw ring does not determine.
 * The first push of a plan compiles the plan-specialised kernel with NVRTC (seconds to a minute, growing with
 * ndm*nchan) and allocates the rings (see nsfrb_plan_create); a compile failure returns NSFRB_ECUDA with
 * the compiler log.  Compiled kernels are cached on disk (NSFRB_JIT_CACHE=<dir>, default /tmp/nsfrb_jit_cache_<uid>, private to the user;
 * NSFRB_JIT_CACHE=0 disables).  nsfrb_plan_prepare(plan, NSFRB_PREPARE_STREAM, chunk_nt) does both ahead of time.  A chunk longer
 * than any before it recompiles the kernel for that length (a stream synchronisation; prepare with the longest chunk to avoid it).
 * Stored samples are kept relative to a per-(channel, pixel) reference level, the median of the first chunk after a reset; the
 * float32 path holds its 1e-4 tolerance while data stay within ~1e3 sigma of it (R32).
 * Non-finite samples: results of the (pixel, trial) series that contain one are unspecified while it is in the ring; once it has
 * left, the carried sums are rebuilt from the ring and the series is exact again (no nsfrb_stream_reset needed).  The same holds
 * for a finite sample of enormous magnitude (R31).
 */
int nsfrb_stream_push(nsfrb_plan *plan, const float *chunk, int chunk_nt, void *stream,
                      float *snr_map, int32_t *argmax,
                      nsfrb_cand *cands, uint32_t cand_capacity, uint32_t *ncands);

/*
 * Optional cube outputs of the real-time path ("the S/N and TOA for all pixels, widths and DMs" are
 * kept for post-processing).  After this call every nsfrb_stream_push also writes, on its stream,
 *   snr_cube  device, [ndm][nwidth][npix] float32: max over this push's windows of S(k, j, t); -INFINITY where the
 *             (dm, width) has no window yet (or never: width longer than the ring)
 *   toa_cube  device, same shape, int32: the window start attaining it (smallest on ties), absolute like argmax's t;
 *             -1 where no window exists
 * in the caller's dm_list / width_list order (pixel-contiguous, like the input).  Trials whose delay vector repeats an
 * earlier one repeat its planes.  Pass two NULLs to switch the outputs off.  The caller owns both buffers.  The first
 * push after switching the outputs on compiles a second variant of the plan's kernel (seconds, cached).
 */
int nsfrb_stream_set_cubes(nsfrb_plan *plan, float *snr_cube, int32_t *toa_cube);

/*
 * Running standard deviation ("normalized by the running standard deviation", L180; SURVEY.md 8(f) NEXT 1,
 * second part; reading R30): besides snr_map/argmax (normalised by this push's own sigma_k, O5), every later push
 * also writes the maps normalised by a standard deviation carried across pushes.  Per (pixel, DM trial):
 *     v_0 = sigma_0^2,   v_n = (1 - alpha) v_{n-1} + alpha sigma_n^2      (sigma_n = this push's sigma_k; a trial
 *     S_run(k,j,t) = (B_j(t) - w_j mu_k) / (sqrt(v_n) sqrt(w_j))           without a valid sample keeps its state)
 * (S_run = 0 where v_n = 0), reduced over (k, j, t) exactly like O6.  A pulse inflates only a fraction alpha of the
 * normalisation of its own push (the bias of L130).  alpha = 1 reproduces snr_map/argmax.
 *   alpha        in (0, 1]
 *   snr_map_run  device, [npix] float32;  argmax_run  device, [3][npix] int32 (layout and conventions of
 *                snr_map/argmax); both NULL switch the mode off.  The caller owns both buffers.
 * The running variance lives in the plan; it restarts with this call and with nsfrb_stream_reset.  The mode uses the
 * per-(trial, width) maxima of nsfrb_stream_set_cubes (the library keeps its own cubes, 8*ndm*nwidth*npix bytes, if the
 * caller registered none) and adds one small launch per push.
 */
int nsfrb_stream_set_running_sigma(nsfrb_plan *plan, double alpha, float *snr_map_run, int32_t *argmax_run);

/* Forget all pushed samples; the plan can be used for nsfrb_search again. */
int nsfrb_stream_reset(nsfrb_plan *plan);

/*
 * Same calls with HOST buffers (pinned memory recommended): the library copies the input
 * host->device, runs the search, copies snr_map/argmax/cands/ncands device->host on
 * `stream` and synchronises it before returning.  Staging buffers belong to the plan.
 * nsfrb_search_host never holds a device copy of the whole cube: it walks the image in pixel batches,
 * copying batch i+1 (a strided block of cube_host: nchan*nt rows of `batch` pixels) on an internal copy stream while batch
 * i is searched; with pinned memory the call is bound by the host link (23.75 GB of C3 at ~55 GB/s: 0.43 s).
 */
int nsfrb_search_host(nsfrb_plan *plan, const float *cube_host, void *stream,
                      float *snr_map_host, int32_t *argmax_host,
                      nsfrb_cand *cands_host, uint32_t cand_capacity, uint32_t *ncands_host);
int nsfrb_stream_push_host(nsfrb_plan *plan, const float *chunk_host, int chunk_nt, void *stream,
                           float *snr_map_host, int32_t *argmax_host,
                           nsfrb_cand *cands_host, uint32_t cand_capacity, uint32_t *ncands_host);

/*
 * Pipelined variant of nsfrb_stream_push_host for back-to-back chunks: the call enqueues the host->device copy of
 * the chunk on a copy stream owned by the plan, the push (nsfrb_stream_push) on a compute stream owned by the plan
 * once the copy has landed, and the device->host copies of snr_map / argmax / ncands and of all cand_capacity
 * candidate records into the caller's buffers -- and returns without waiting.  The copy of chunk i+1 overlaps the
 * search of chunk i.  Two pushes may be in flight (two staging slots): a third call first waits for the oldest.
 *   chunk_host and the four output buffers must stay valid and untouched until nsfrb_stream_wait (or the second
 *   following call) returns; use page-locked memory, otherwise the copies are staged by the driver and do not overlap.
 *   Different pushes in flight need different output buffers.
 * nsfrb_stream_wait blocks until every push in flight has delivered its outputs.  Do not mix with
 * nsfrb_stream_push / nsfrb_stream_push_host / nsfrb_stream_reset on the same plan without an nsfrb_stream_wait (and,
 * for the device-pointer variant, a synchronisation of the caller's stream) in between.
 */
int nsfrb_stream_push_host_async(nsfrb_plan *plan, const float *chunk_host, int chunk_nt, float *snr_map_host,
                                 int32_t *argmax_host, nsfrb_cand *cands_host, uint32_t cand_capacity,
                                 uint32_t *ncands_host);
int nsfrb_stream_wait(nsfrb_plan *plan);

/* Release everything the plan owns.  NULL is a no-op returning 0. */
int nsfrb_plan_destroy(nsfrb_plan *plan);

/* Copy the integer delay table to host memory out[ndm][nchan] (bit-exact parity check). */
int nsfrb_plan_get_delays(const nsfrb_plan *plan, int32_t *out);

/* Fill *info. */
int nsfrb_plan_get_info(const nsfrb_plan *plan, nsfrb_plan_info *info);

/* Number of kernel launches the last nsfrb_search / nsfrb_stream_push enqueued. */
int nsfrb_plan_last_launches(const nsfrb_plan *plan);

/*
 * How the real-time path of this plan holds its data, for harnesses that report traffic:
 *   0  no streaming state yet (no push, no NSFRB_PREPARE_STREAM)
 *   1  raw ring only: every push dedisperses the rows it marches over
 *   2  raw ring + dedispersed history: D_u(t) of every unique trial is formed once, when the sample arrives
 *   3  as 2, plus the sums of the history's 8-sample blocks (ring length a multiple of 8): the default where it fits
 * Mode 2/3 take nuniq/nchan times the raw ring's memory again; where that exceeds half of the free device memory at the
 * first push (or with NSFRB_STREAM_DHIST=0) the plan runs in mode 1.  Results are the same in every mode (S-rules).
 */
int nsfrb_stream_mode(const nsfrb_plan *plan);

/*
 * Per-kernel device timing for harnesses.  With profiling on, every call records CUDA events
 * on its stream around each kernel it enqueues.  nsfrb_plan_get_kernel_ms waits for the last
 * call's events and writes the milliseconds of out[0] = layout kernel (transpose or ring push),
 * out[1] = search kernel, out[2] = finalize kernel, out[3] = candidate compaction.
 */
int nsfrb_plan_set_profiling(nsfrb_plan *plan, int on);
int nsfrb_plan_get_kernel_ms(nsfrb_plan *plan, float out[4]);

/*
 * Time binning for the paper's longer timescales (images are binned x5 to 0.67 s and x75 to
 * 10.05 s and searched again with the same widths; by footnote 12, L98, a plan created with 5*tsamp and 5*dm has
 * the same shift table).  out[c][u][p] = sum_{i<factor} cube[c][u*factor+i][p] for u < nt/factor (integer
 * division; trailing samples are dropped; a sum, not a mean -- the S/N is scale-free).
 *   cube  device, [nchan][nt][npix] float32, read only;  out  device, [nchan][nt/factor][npix], must not alias cube
 * Asynchronous on `stream`.  NSFRB_EINVAL for null pointers or non-positive sizes/factor.
 */
int nsfrb_bin_time(const float *cube, int nchan, int nt, int64_t npix, int factor, float *out, void *stream);

/*
 * Per-pixel median subtraction ("Data is first median subtracted in each pixel"; SURVEY.md 8(f) NEXT 1,
 * first part; reading R29).  For every (channel c, pixel p): m = the median of cube[c][0..nt-1][p] -- the middle
 * element of the sorted series, for even nt the mean of the two middle elements computed in float64 and rounded once
 * to float32 -- and out[c][t][p] = cube[c][t][p] - m (float32).  Inputs must be finite (no NaN).  Under the path's
 * per-(pixel, DM) mean subtraction (O3) this step changes no S/N beyond rounding; it is provided as the first stage
 * of the paper's robust-baseline variant.
 *   cube    device, [nchan][nt][npix] float32, read only unless out == cube
 *   out     device, same shape; may be the same pointer as cube (in place), must not overlap it otherwise
 *   median  device, [nchan][npix] float32, written (may be NULL)
 * Asynchronous on `stream`; one launch.  NSFRB_EINVAL for null pointers, non-positive sizes, nchan > 65535 or
 * nt > 65535 (16-bit histogram counters).
 */
int nsfrb_median_subtract(const float *cube, int nchan, int nt, int64_t npix, float *out, float *median, void *stream);

/*
 * Post-search candidate selection (readings R25-R28 in DESIGN.md).
 *
 * nsfrb_psf_mask: "the PSF is thresholded at the 90th percentile to make a binary mask".  The percentile value is
 * v[lo] + (r - lo)*(v[lo+1] - v[lo]) with v = the PSF elements in ascending order, r = percentile/100*(mh*mw - 1),
 * lo = floor(r), evaluated in float64; mask[i] = 1 where (double)psf[i] > value, else 0.
 *   psf    device, [mh][mw] float32, finite values, read only
 *   mask   device, [mh][mw] uint8, written
 *   value  device, one float64, written (may be NULL)
 * Asynchronous on `stream`; one launch.  NSFRB_EINVAL for null pointers, non-positive sizes, a percentile outside
 * [0, 100] or more than 2^31-1 elements.
 *
 * nsfrb_cluster: "Standard post-processing is limited to the 10 highest S/N candidates ... [the mask] is centered
 * on each candidate in turn.  This candidate is treated as the central PSF lobe, and any other candidates within the
 * binary mask are identified as possible sidelobes.  The weighted mean S/N is computed over the central and sidelobe
 * candidate S/Ns.  After repeating with each candidate, the maximum S/N is identified and its central lobe
 * candidate's width, DM, position, and TOA are taken as the final, most-likely candidate."
 *   Candidates: the pixels with snr_map > the plan's threshold (strict); the `topn` highest, equal S/N -> smaller
 *   pixel index; n_found <= topn of them exist.  For centre i (rank order, best first) a candidate j at offset
 *   (dx, dy) = (x_j - x_i, y_j - y_i) is a member if j == i, or if (mh/2 + dy, mw/2 + dx) lies inside the PSF array
 *   and the mask is set there; its weight is the PSF value there (psf[mh/2][mw/2] for the centre).
 *   wsnr[i] = sum_j w_j*snr_j / sum_j w_j over the members in rank order, float64, each operation rounded once.
 *   best = the i with the largest wsnr (equal -> smaller i), -1 if n_found == 0.
 *   snr_map  device, [ny][nx] float32, and  argmax  device, [3][npix] int32: outputs of nsfrb_search /
 *            nsfrb_stream_push of this plan (or anything of that layout); read only
 *   psf, mask  device, [mh][mw] float32 / uint8 (as written by nsfrb_psf_mask); psf[mh/2][mw/2] must be > 0
 *   topn     1..32
 *   top      device, [topn] nsfrb_cand: the candidates in rank order; entries >= n_found are (-1,-1,-1,-1,0)
 *   wsnr     device, [topn] float64;  members  device, [topn] int32 (member counts; 0 beyond n_found)
 *   result   device, [2] int32: n_found, best
 * Asynchronous on `stream`; one launch; the first call allocates a small workspace in the plan.  Calls on one plan
 * must be stream-ordered (as for nsfrb_search).  NSFRB_EINVAL for null arguments or sizes out of range.
 */
int nsfrb_psf_mask(const float *psf, int mh, int mw, double percentile, uint8_t *mask, double *value, void *stream);
int nsfrb_cluster(nsfrb_plan *plan, const float *snr_map, const int32_t *argmax, const float *psf,
                  const uint8_t *mask, int mh, int mw, int topn, nsfrb_cand *top, double *wsnr, int32_t *members,
                  int32_t *result, void *stream);

/*
 * nsfrb_cluster for callers that may not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc).  Same computation and outputs as nsfrb_cluster (readings R25-R28), but
 * no plan is needed -- nx, ny and the threshold are arguments -- and the kernel's workspace is a fixed array in the
 * library's device image (38 144 bytes, held by every GPU that loads the library until the process exits).  The call
 * makes no cudaMalloc / cudaFree and no allocating library call: one 256-byte cudaMemsetAsync and one kernel launch on
 * `stream`, on the CURRENT device (the first call on a device also looks the array's address up).
 *   Limits: nx*ny <= 16 777 216 pixels, 1 <= topn <= 32; beyond them NSFRB_EINVAL with a message naming the limit.
 *   All calls in the process share the workspace: calls on one GPU must be stream-ordered (or otherwise not overlap);
 *   two that run concurrently race.  The workspace keeps the previous call's contents; the call clears what it needs.
 *   Arguments and outputs as nsfrb_cluster; snr_map is [ny][nx], argmax [3][nx*ny].
 */
int nsfrb_cluster_static(int nx, int ny, float threshold, const float *snr_map, const int32_t *argmax,
                         const float *psf, const uint8_t *mask, int mh, int mw, int topn, nsfrb_cand *top,
                         double *wsnr, int32_t *members, int32_t *result, void *stream);

/*
 * Harness access to the plan-specialised real-time kernel: for the plan the first ten
 * arguments describe (as nsfrb_plan_create) and a first chunk of chunk_nt samples, writes either the CUDA
 * source the library compiles at the first nsfrb_stream_push (want_cubin = 0) or its sm_100a cubin
 * (want_cubin = 1, compiled with NVRTC) to out[capacity] (host) and the byte count to *needed; call with
 * out = NULL to size the buffer.  variant = NULL or "" selects the default tile shape, else
 * "KK,GPC,SEG,TT[,MINB]".  Needs no CUDA device.
 */
int nsfrb_jit_stream_kernel(int nx, int ny, int nchan, int nt, const double *freqs_GHz, double tsamp_s,
                            const double *dm_list, int ndm, const int32_t *width_list, int nwidth,
                            int chunk_nt, const char *variant, int want_cubin,
                            char *out, size_t capacity, size_t *needed);

/* The same for the plan-specialised offline kernel k_search3 (compiled at the first nsfrb_search of a plan with at
 * most 32 usable widths; NSFRB_SEARCH_JIT=0 selects the generic k_search instead). */
int nsfrb_jit_search_kernel(int nx, int ny, int nchan, int nt, const double *freqs_GHz, double tsamp_s,
                            const double *dm_list, int ndm, const int32_t *width_list, int nwidth,
                            int want_cubin, char *out, size_t capacity, size_t *needed);

/*
 * Upstream imaging (PAPER.md:L55, L61 fn. 10, L67; readings I1-I6 in DESIGN.md): fringe-stopped
 * visibilities of one sub-band -> one n x n image per time sample, ready to be a channel plane of a search chunk.
 *   "grids visibilities with baseline lengths b > b_min = 20 m from the dense 82-antenna 'core' (b < b_max = 485 m) to a
 *    175 x 175-pixel UV-grid ... The two visibility polarizations are summed, then approximately uniform weighting (Briggs
 *    robustness parameter R = -2) is applied to accumulate visibilities, and a 2-dimensional inverse-FFT is applied" (L55);
 *   "ifftshift ... np.fft.ifft2 ... ifftshift" (L61); "Each of the 8 channels are imaged individually, then summed" (L67).
 * Definition.  For channel c and baseline b with bmin < |uv_m[b]| < bmax:  (fu, fv) = floor(uv_m[b] * f_c / c_light * n *
 * pixel_rad + 0.5) (nearest UV cell, offsets from grid index n/2; baselines whose cell or its mirror image falls off the grid
 * are dropped); natural weight 1; W_k = number of visibilities in cell k counting every visibility at (fu, fv) and (-fu, -fv);
 * Briggs weight w = 1 / (1 + W_k f^2), f^2 = (5 * 10^-robust)^2 / (sum_k W_k^2 / sum_i 1).  The channel's grid holds
 * w (V0 + V1) at (fu, fv) and its conjugate at (-fu, -fv); channel image = Re(ifftshift(ifft2(ifftshift(grid)))) * n^2 /
 * (2 sum w) (a unit point source at the phase centre has value 1 at pixel (x0, x0), x0 = n - n/2: the pixel the final
 * ifftshift moves index 0 to); out = the sum of the channel images.  x runs with u (l), y with v (m); out[t][y][x].
 *
 * nsfrb_imager_create: all of the above that does not depend on the data, in float64 on the host; small tables go to the
 *   current device.  uv_m host [nbase][2] metres (east, north); freqs_GHz host [nchan].  2 <= n <= 2048.
 * nsfrb_imager_image:  vis device, [nt][nchan][nbase][2 pol] complex64 as (re, im) float32 pairs (the paper's 14.9 MB
 *   buffer for nt = 25), 16-byte aligned, read only;  out device, [nt][n*n] float32, written.  One launch on `stream`,
 *   asynchronous.  With out = chunk + subband * nt * n * n the result is one channel plane of an nsfrb_stream_push chunk.
 * nsfrb_imager_get_table: cells host [nchan][nbase][2] int32 and weights host [nchan][nbase] float64 (0 = not gridded), for
 *   bit-exact parity of the integer part.
 * Errors: NSFRB_EINVAL (null, sizes, non-finite parameters, misaligned vis), NSFRB_ENOMEM, NSFRB_ECUDA.
 */
typedef struct nsfrb_imager nsfrb_imager;
int nsfrb_imager_create(nsfrb_imager **out, int n, double pixel_rad, const double *uv_m, int nbase,
                        const double *freqs_GHz, int nchan, double bmin_m, double bmax_m, double robust);
int nsfrb_imager_image(nsfrb_imager *imager, const float *vis, int nt, float *out, void *stream);
int nsfrb_imager_get_table(const nsfrb_imager *imager, int32_t *cells, double *weights);
int nsfrb_imager_destroy(nsfrb_imager *imager);

/*
 * Measured on-chip ceilings of the current device, for the offline roofline ("the builder writes two
 * microbenchmarks (FADD/FMNMX chain; conflict-free LDS stream) and uses the achieved numbers").  Runs one short
 * kernel per instruction mix on every SM (about 0.1 s in all with iters = 2000); synchronises `stream`.
 *   nsfrb_peaks_count()   number of tests;  nsfrb_peaks_name(i)  its name (static string, "" out of range):
 *     fadd, fmnmx, fmnmx3, ffma, fadd2_fmnmx3_pair (two differences + one 3-input maximum, the search's cell pair),
 *     viaddmnmx, iadd  -- lane-operations issued;   lds32, lds128 -- conflict-free 4-byte words out of shared memory
 *   per_s        host, [count] float64: operations (or words) per second over the whole GPU, timed with CUDA events
 *   per_clk_sm   host, [count] float64: the same per SM clock and SM, from clock64 spans of the slowest CTA
 * NSFRB_EINVAL for null pointers or iters < 1; NSFRB_ECUDA on a CUDA error.
 */
int nsfrb_peaks_count(void);
const char *nsfrb_peaks_name(int test);
int nsfrb_measure_peaks(int iters, double *per_s, double *per_clk_sm, void *stream);

/* Thread-local text of the last error; never NULL. */
const char *nsfrb_last_error(void);

/* "major.minor (build tag)". */
const char *nsfrb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NSFRB_H */
