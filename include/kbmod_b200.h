/*
 * kbmod_b200.h -- C ABI of libkbmod_b200.so: the data-parallel hot path of the KBMOD
 * shift-and-stack moving-object search as extended by Smotherman et al. (arXiv 2109.03296),
 * hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Citations are "PAPER.md:L<line>" (/root/reference/PAPER.md, the text of the paper) plus the
 * section / equation the line falls in.  Readings of points the paper leaves open are the
 * R-numbers of DESIGN.md.
 *
 * Conventions (all entry points)
 *   - extern "C", plain pointers and sizes.  `d_` = DEVICE pointer (current CUDA device),
 *     `h_` = HOST pointer.  Host arrays are consumed before the call returns.
 *   - The library never allocates or frees device memory: every device buffer (inputs,
 *     outputs, workspace) is caller-owned.  (The *_host convenience calls take a caller-owned
 *     device arena for the same reason.)  Host-side state exists in two places only, both
 *     with an owner: a kbmod_plan (created / destroyed by the caller) and the per-thread
 *     conveniences listed at kbmod_release_thread_state(), which frees them.
 *   - All kernels are enqueued on `stream` (a cudaStream_t passed as void*; NULL = the legacy
 *     default stream).  Calls return without synchronising unless stated.
 *   - Layouts are C-contiguous with x fastest: stacks are [T][H][W]; the psi/phi stack is
 *     [T][H][W][2] float (psi, phi interleaved, i.e. a CUDA float2 per pixel).
 *   - Every function returns an int status: KBMOD_OK (0) or a negative error code;
 *     kbmod_last_error() gives a thread-local message for the last failure.
 *   - Limits: T <= 64 epochs, K <= 32 results per pixel, PSF side k odd and <= 31,
 *     stamp radius <= 15, T*H*W < 2^31 pixels per stack, W, H <= 32767, and for a search
 *     (T + 1) * (W + pad_x) * (H + pad_y) < 2^32 where pad = the largest displacement of the
 *     velocity list on each side, clamped to the image size.  Outside -> KBMOD_ERR_UNSUPPORTED.
 *   - There is no CPU fallback: without a CUDA device every compute entry point fails with
 *     KBMOD_ERR_CUDA.
 */
#ifndef KBMOD_B200_H
#define KBMOD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KBMOD_OK 0
#define KBMOD_ERR_INVALID_ARG (-1) /* null pointer, non-positive size, inconsistent arguments      */
#define KBMOD_ERR_UNSUPPORTED (-2) /* a documented limit is exceeded (see above)                   */
#define KBMOD_ERR_WORKSPACE (-3)   /* workspace_bytes < kbmod_search_workspace_bytes(...)          */
#define KBMOD_ERR_CUDA (-4)        /* a CUDA runtime / driver call failed (message has the detail) */

#define KBMOD_MAX_T 64
#define KBMOD_MAX_K 32
#define KBMOD_MAX_PSF 31
#define KBMOD_MAX_STAMP_RADIUS 15

/* Which search kernel kbmod_search runs.  Both give the same results. */
#define KBMOD_ALGO_AUTO 0   /* pruned when min_lh is finite and sigma-G is on, else direct       */
#define KBMOD_ALGO_DIRECT 1 /* every trajectory gets the full sigma-G evaluation                 */
#define KBMOD_ALGO_PRUNED 2 /* exact upper bound from shared-memory tiles first, full evaluation
                               only for trajectories whose bound reaches the threshold           */

/* sigma-G filter + selection parameters.  kbmod_default_params() fills the paper's values. */
typedef struct {
    int sigmag_enable; /* 1: apply the in-line sigma-G lightcurve filter (s3.2)   */
    float pct_lo;      /* 25  lower percentile  (s3.1)                                  */
    float pct_hi;      /* 75  upper percentile                                        */
    float sigmag_coeff;/* 0.7413  sigma_G = coeff * (P_hi - P_lo)  (Eq. 5)              */
    float n_sigma;     /* 2   keep points within +- n_sigma * sigma_G of the median    */
    int filter_on;     /* 0: filter the flux lightcurve psi/phi; 1: the likelihood lightcurve
                          psi/sqrt(phi)  ("likelihood and/or flux values"; reading R9)   */
    float min_lh;      /* keep a trajectory iff its recomputed likelihood L' >= min_lh
                          (10); -INFINITY keeps everything                              */
    int min_obs;       /* minimum number of valid epochs BEFORE filtering (reading R8)  */
    int K;             /* results kept per start pixel (8)                              */
    int algo;          /* KBMOD_ALGO_*                                                                 */
    int pct_interp;    /* 0: percentiles are nearest-rank order statistics (reading R10, the default);
                          1: linear interpolation between the two bracketing order statistics, as
                          numpy.percentile(method="linear") (reading R23; PAPER.md:L117 leaves it open)     */
} kbmod_search_params;

/* Host-only: where the three percentiles (pct_lo, 50, pct_hi) of n valid samples sit in the ascending sort, as the
 * kernels use them: h_k[i] = index k; h_g[i] < 0: the percentile is s[k] (nearest rank, or a clamped end);
 * h_g[i] = g >= 0: it is s[k] + g (s[k+1] - s[k]) (pct_interp = 1). */
int kbmod_percentile_ranks(const kbmod_search_params* p, int n, int* h_k, float* h_g);

/* Fills *p with the paper's operating point: sigma-G on, 25/75, 0.7413, n=2, flux lightcurve,
 * min_lh=10, min_obs=1, K=8, algo=AUTO, nearest-rank percentiles. */
void kbmod_default_params(kbmod_search_params* p);

/* ---------------------------------------------------------------------------------------------
 * (a1) psi/phi preparation.  PAPER.md:L79 (s3): "KBMOD generates images of likelihood (Psi_i)
 * and variance (Phi_i) ... as described in Whidden et al. (2019)"; masks and variance planes are
 * part of the input.  Reading R1-R4:
 *     w(x,y)   = 1/var(x,y) if the pixel is on-image, mask==0, var>0, img and var finite; else 0
 *     Psi(x,y) = sum_{j,i} P[j][i] * img(x+i-r, y+j-r) * w(x+i-r, y+j-r)        (correlation)
 *     Phi(x,y) = sum_{j,i} P[j][i]^2 * w(x+i-r, y+j-r),        r = k/2
 * An output pixel whose own centre pixel has w == 0 is invalid and is written as (0, 0).
 *   d_img, d_var  [T][H][W] float32          d_mask  [T][H][W] uint8, non-zero = bad; may be NULL
 *   h_psf         [n_psf][k][k] float32 on the HOST; n_psf is 1 (shared) or T (per epoch); k odd
 *   d_psiphi      out, [T][H][W][2] float32
 * float32 arithmetic (FMA accumulation); agrees with the double-precision definition to
 * 1e-5 * sum|P I w| (psi) and 1e-5 * Phi (phi). */
int kbmod_prepare_psi_phi(const float* d_img, const float* d_var, const uint8_t* d_mask, int T, int H, int W,
                          const float* h_psf, int n_psf, int k, float* d_psiphi, void* stream);

/* ---------------------------------------------------------------------------------------------
 * (a2) displacement table, host only (no GPU needed).  PAPER.md:L79-L81: the images are
 * "shifted along a potential asteroid trajectory" by "pointer arithmetic"; reading R5/R18:
 *     dx[v][t] = floor( (double)vx[v] * (times[t]-times[0]) + 0.5 )     (round half up)
 * multiply and add separately rounded in IEEE double.  The position of trajectory (x0,y0,v) at
 * epoch t is (x0+dx[v][t], y0+dy[v][t]).   h_dx, h_dy: out, [n_vel][T] int32. */
int kbmod_displacements(const double* h_times, int T, const float* h_vx, const float* h_vy, int n_vel,
                        int32_t* h_dx, int32_t* h_dy);

/* ---------------------------------------------------------------------------------------------
 * (a3)-(a5) the search: gather + in-line sigma-G + per-pixel top-K.
 * PAPER.md:L79 (Psi_coadd = sum Psi_i, Phi_coadd = sum Phi_i, nu = Psi_coadd/sqrt(Phi_coadd)),
 * L81, L93-L117 (s3.1, Eq. 1-5), L123, L127-L137 (s3.2).  For every start pixel (x0,y0) in
 * [0,W)x[0,H) and every velocity v in [0,n_vel):
 *   1. gather (psi_t, phi_t) at (x0+dx[v][t], y0+dy[v][t]); a sample is valid iff on-image and
 *      phi_t > 0; n = number of valid samples; if n < max(1,min_obs) the trajectory has no result;
 *   2. if sigmag_enable: f_t = psi_t/phi_t (filter_on=0) or psi_t/sqrt(phi_t) (filter_on=1) in
 *      IEEE float32; s = ascending sort of the n valid f; P_q = s[ceil(q*n/100)-1] (nearest rank,
 *      clamped to [0,n-1]; R10) -- or, with pct_interp, s[k] + g (s[k+1] - s[k]) at h = (n-1) q / 100,
 *      k = floor(h), g = h - k, three separately rounded float32 operations (R23);
 *      sigma_G = coeff*(P_hi-P_lo); kept = { t valid :
 *      P_50 - n_sigma*sigma_G <= f_t <= P_50 + n_sigma*sigma_G } (one pass, inclusive bounds,
 *      each float32 operation separately rounded; R11-R13).  Else kept = valid;
 *   3. L' = sum_kept psi / sqrt(sum_kept phi), flux' = sum_kept psi / sum_kept phi (float32);
 *      the trajectory is dropped if !(L' >= min_lh);
 *   4. per start pixel keep the K survivors with the largest L' (ties: lower velocity index),
 *      sorted descending.
 * Outputs, each [H][W][K]: d_lh (L'), d_flux (flux'), d_vel_idx, d_n_obs (= |kept|).  Unfilled
 * slots hold lh=-INFINITY, flux=0, vel_idx=-1, n_obs=0.
 *   d_psiphi   [T][H][W][2] float32 (kbmod_prepare_psi_phi's output; not modified)
 *   h_times    [T] double, days, any zero point, any order (R18)
 *   h_vx, h_vy [n_vel] float32, px/day
 *   d_workspace caller-owned scratch, 256-byte aligned; contents undefined on entry.  Its size depends on the
 *               velocity list (the search pads its working copy of the stack by the largest displacement):
 *               kbmod_search_workspace_bytes_for(...) gives the exact need, kbmod_search_workspace_bytes(...) an
 *               upper bound valid for any list of n_vel velocities (the image padded by its own size on every
 *               side).  On exit the workspace holds the padded stack and the offset table that
 *               kbmod_search_unfiltered_lh reads.
 * kbmod_search does the host-side planning (displacement table, padded-stack geometry, choice of kernel, velocity
 * grouping) once per geometry: the plan is kept per host thread and reused while T, H, W, the row band, the times,
 * the velocities and the parameters are unchanged (kbmod_plan_* below is the same thing with an explicit owner).
 * The tables go to the workspace with ONE cudaMemcpyAsync from pinned host memory, so the call does not wait for
 * earlier work on the stream.  Test hook: the environment variable KBMOD_B200_QUEUE_CAP=<entries> shrinks the
 * internal survivor queue of the pruned kernel (results are unaffected; it exercises the overflow path). */
size_t kbmod_search_workspace_bytes(int T, int H, int W, int n_vel, const kbmod_search_params* p);
size_t kbmod_search_workspace_bytes_for(int T, int H, int W, const double* h_times, const float* h_vx, const float* h_vy,
                                        int n_vel, const kbmod_search_params* p, int row_begin, int row_end);
int kbmod_search(const float* d_psiphi, int T, int H, int W, const double* h_times, const float* h_vx,
                 const float* h_vy, int n_vel, const kbmod_search_params* p, float* d_lh, float* d_flux,
                 int32_t* d_vel_idx, int32_t* d_n_obs, void* d_workspace, size_t workspace_bytes, void* stream);

/* The same search restricted to the start pixels of the row band [row_begin, row_end) (trajectories are
 * independent, so one CCD shards over GPUs by start-pixel row bands -- every GPU holds the whole psi/phi stack,
 * results concatenate, no merge).  Outputs are [row_end - row_begin][W][K]; a band's results equal the same rows of
 * the full search bit for bit. */
int kbmod_search_rows(const float* d_psiphi, int T, int H, int W, const double* h_times, const float* h_vx,
                      const float* h_vy, int n_vel, const kbmod_search_params* p, int row_begin, int row_end, float* d_lh,
                      float* d_flux, int32_t* d_vel_idx, int32_t* d_n_obs, void* d_workspace, size_t workspace_bytes,
                      void* stream);

/* Unfiltered sum-LH beside sum-LH' (s4.1: the single-trajectory variant "computes the likelihoods
 * along a single trajectory then runs the ... filtering"; L181 quotes both for the recovered objects): for every
 * result slot with vel_idx >= 0, L = sum psi / sqrt(sum phi) over ALL valid epochs of that trajectory -- no
 * sigma-G clip, no threshold; empty slots get -INFINITY.  Reads the padded stack the last kbmod_search of this
 * host thread left in `d_workspace` (so: same thread, same workspace, after that search on the same stream).
 *   d_vel_idx  [rows][W][K] int32 (kbmod_search's output)      d_lh_raw  out [rows][W][K] float32 */
int kbmod_search_unfiltered_lh(const void* d_workspace, const int32_t* d_vel_idx, float* d_lh_raw, void* stream);

/* ---------------------------------------------------------------------------------------------
 * The search with an explicit plan (the multi-CCD / multi-stream form; 2580 searches = 43 pointing
 * groups x 60 CCDs, one grid and one set of epoch times per group).  A plan holds everything that depends on the
 * geometry alone -- host memory only (pinned), immutable after creation -- so the searches of all CCDs of a
 * pointing group, on any number of streams, share ONE plan; each search needs its own workspace of
 * kbmod_plan_workspace_bytes().  kbmod_plan_search enqueues: one table upload, the padded-stack build, the
 * search kernels, the key -> output pass; it never synchronises and never touches pageable host memory.
 * The table upload (a few MB, host to device from pinned memory) is ordered by the device's copy engine: behind a large
 * host-to-device copy that is in flight on another stream it waits for that copy, and the search with it.
 * kbmod_pipeline_host_batch, which has such copies in flight by design, uploads the tables once per call instead.
 *   row_begin, row_end   the band of start rows this plan searches (0, H for the whole image)
 * kbmod_plan_info fills h_out[10]: kernel used (KBMOD_ALGO_DIRECT / PRUNED), velocity groups, bytes staged into shared
 * memory per trajectory-epoch evaluation, share of (tile, group, epoch) region loads that lie off the image, padded
 * stack width and height, 1 if the velocity list was too scattered for the pruned kernel, bytes of the table blob,
 * shared-memory gathers per nominal evaluation before off-image skipping (< 1: epochs at which a whole velocity group
 * has one displacement are gathered once per pixel), workspace bytes. */
typedef struct kbmod_plan kbmod_plan;
int kbmod_plan_create(int T, int H, int W, const double* h_times, const float* h_vx, const float* h_vy, int n_vel,
                      const kbmod_search_params* p, int row_begin, int row_end, kbmod_plan** out);
size_t kbmod_plan_workspace_bytes(const kbmod_plan* plan);
int kbmod_plan_info(const kbmod_plan* plan, double* h_out);
int kbmod_plan_search(kbmod_plan* plan, const float* d_psiphi, float* d_lh, float* d_flux, int32_t* d_vel_idx,
                      int32_t* d_n_obs, void* d_workspace, size_t workspace_bytes, void* stream);
int kbmod_plan_unfiltered_lh(const kbmod_plan* plan, const void* d_workspace, const int32_t* d_vel_idx, float* d_lh_raw,
                             void* stream);
void kbmod_plan_destroy(kbmod_plan* plan); /* waits for the plan's last table upload, then frees it */

/* Frees everything the library keeps per host thread: the cached plan of kbmod_search / kbmod_pipeline_host*, the
 * CUDA events of kbmod_search_phase_timing, the two copy streams and six events of kbmod_pipeline_host_batch.
 * Safe at any time (it waits for the cached plan's last upload); later calls recreate what they need. */
int kbmod_release_thread_state(void);

/* Host-only view of the pruned kernel's plan for a geometry (no GPU needed; what `-m "not gpu"` tests check):
 * h_out[0] = 1 if the velocity list is too scattered for the pruned kernel (AUTO then runs the direct one), h_out[1] =
 * bytes staged into shared memory per trajectory-epoch evaluation, h_out[2] = number of velocity groups, h_out[3] =
 * share of the (tile, group, epoch) region loads that lie off the image and are skipped. */
int kbmod_plan_stats(int T, int H, int W, const double* h_times, const float* h_vx, const float* h_vy, int n_vel,
                     const kbmod_search_params* p, double* h_out);

/* Counters of the last search that used this workspace (a blocking 40-byte read; synchronises the device).
 * h_out[5]: [0] = trajectories fully evaluated (sigma-G run), [1] = trajectories nominally searched (rows*W*n_vel),
 * [2] = kernels launched by the call, [3] = algo actually used, [4] = pruned path only: trajectories whose L'
 * reached min_lh, i.e. the candidates before the per-pixel top-K (PAPER.md:L91 quotes ~10^7 per search); 0 for the
 * direct kernel. */
int kbmod_search_stats(const void* d_workspace, unsigned long long* h_out);

/* Optional timing of the phases of kbmod_search, per host thread (what bench.py's roofline line reads).
 * kbmod_search_phase_timing(1) makes every following search on this thread record CUDA events on its stream
 * between its phases (the library creates and keeps a few cudaEvent_t for this -- no device memory;
 * kbmod_release_thread_state() destroys them).
 * kbmod_search_phase_ms waits for the last timed search and fills h_ms[4] with the milliseconds spent in
 *   [0] padded stack + bound planes, [1] the gather kernel: bound phase of the pruned path / the whole direct kernel,
 *   [2] exact evaluation of the surviving trajectories (pruned only), [3] top-K keys -> output arrays. */
int kbmod_search_phase_timing(int enable);
int kbmod_search_phase_ms(float* h_ms);

/* ---------------------------------------------------------------------------------------------
 * (a6) coadded stamps.  PAPER.md:L141 (s3.3): stamps are coadded by "computing the median pixel
 * value for each pixel along the trajectory"; mean/sum is the earlier variant; 21x21 (L145, L175);
 * reading R17.  For trajectory i and stamp offset (u,v) in [-radius,radius]^2 the samples are
 * img_t(x0+dx_t+u, y0+dy_t+v) over epochs t that are selected (bit t of d_epoch_mask[i], all
 * epochs when d_epoch_mask is NULL), on-image, unmasked and finite.  mean = sum/count;
 * median = middle of the sort (mean of the two middles for an even count); count 0 -> 0.
 *   d_x0,d_y0 [n_traj] int32; d_vx,d_vy [n_traj] float32 (px/day); displacements as in (a2)
 *   d_mean, d_median  out, [n_traj][2r+1][2r+1] float32 (v rows, u columns); either may be NULL */
int kbmod_coadd_stamps(const float* d_img, const uint8_t* d_mask, int T, int H, int W, const double* h_times,
                       const int32_t* d_x0, const int32_t* d_y0, const float* d_vx, const float* d_vy,
                       const uint64_t* d_epoch_mask, int n_traj, int radius, float* d_mean, float* d_median,
                       void* stream);

/* ---------------------------------------------------------------------------------------------
 * Single-trajectory variant (s4.1: "computes the likelihoods along a single
 * trajectory then runs the ... quantile-based filtering").  Steps 1-3 of kbmod_search for an
 * explicit list of trajectories; min_lh and K are ignored.
 *   d_psi_lc, d_phi_lc  out [n_traj][T] float32 (0 where invalid); may be NULL
 *   d_valid, d_kept     out [n_traj] uint64, bit t = epoch t valid / kept; may be NULL
 *   d_lh, d_flux        out [n_traj] float32; n < max(1,min_obs): lh=-INFINITY, flux=0, kept=0 */
int kbmod_eval_trajectories(const float* d_psiphi, int T, int H, int W, const double* h_times,
                            const int32_t* d_x0, const int32_t* d_y0, const float* d_vx, const float* d_vy,
                            int n_traj, const kbmod_search_params* p, float* d_psi_lc, float* d_phi_lc,
                            uint64_t* d_valid, uint64_t* d_kept, float* d_lh, float* d_flux, void* stream);

/* sigma-G on given lightcurves (the paper's post-filter; BASELINE configs[4]).
 * Epoch t of lightcurve i is valid iff d_phi_lc[i][t] > 0.  Steps 2-3 of kbmod_search; min_lh and K are ignored. */
int kbmod_sigmag_filter(const float* d_psi_lc, const float* d_phi_lc, int n_lc, int T,
                        const kbmod_search_params* p, uint64_t* d_kept, float* d_lh, float* d_flux, void* stream);

/* The post-filter with the paper's decision ("reject the trajectory if the recomputed likelihood
 * (sum LH') is less than 10"; ~10^6 such rejections per search in the paper): as kbmod_sigmag_filter, plus
 *   d_pass       out [n_lc] uint8: 1 iff the lightcurve has a result (n_valid >= max(1, min_obs)) and L' >= min_lh
 *   d_survivors  out, nullable: the indices i with d_pass[i] = 1, ascending, compacted to the front ([n_lc] int32)
 *   d_n_pass     nullable (required with d_survivors): 4 uint64 of device scratch; on completion [0] = number of
 *                survivors.  d_kept, d_lh, d_flux may be NULL. */
int kbmod_sigmag_postfilter(const float* d_psi_lc, const float* d_phi_lc, int n_lc, int T,
                            const kbmod_search_params* p, uint64_t* d_kept, float* d_lh, float* d_flux, uint8_t* d_pass,
                            int32_t* d_survivors, uint64_t* d_n_pass, void* stream);

/* The same post-filter for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): results identical to kbmod_sigmag_postfilter, but the
 * scratch -- the pass flags and the counters of the ordered compaction -- is a static device array inside the library:
 * KBMOD_POSTFILTER_STATIC_MAX_LC flag bytes + 256 B (4 MiB + 256 B on every GPU that loads the library, until exit).
 * The call allocates nothing (no cudaMalloc / cudaFree, no allocating library routine); it enqueues two 8/32-byte
 * memsets and two kernels on `stream` and returns without synchronising.
 *   d_survivors    out [n_lc] int32: indices with a result and L' >= min_lh, ascending, compacted to the front
 *   d_n_survivors  out, 1 uint64 (device): their number
 *   d_kept, d_lh, d_flux  out, nullable, as in kbmod_sigmag_filter
 * n_lc > KBMOD_POSTFILTER_STATIC_MAX_LC returns KBMOD_ERR_WORKSPACE (split the list, or use kbmod_sigmag_postfilter).
 * Every call on a device shares the one array, which keeps the previous call's contents (the call clears what must
 * start at zero): calls that overlap on the GPU -- different streams with no ordering between them -- race. */
#define KBMOD_POSTFILTER_STATIC_MAX_LC (1 << 22)
int kbmod_sigmag_postfilter_static(const float* d_psi_lc, const float* d_phi_lc, int n_lc, int T,
                                   const kbmod_search_params* p, uint64_t* d_kept, float* d_lh, float* d_flux,
                                   int32_t* d_survivors, uint64_t* d_n_survivors, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Central-moment stamp filter, the step behind the coadd (s3.3): "we computed the central moments
 * of postage stamps for candidate trajectories.  Stamps were rejected if they did not have central moments that
 * were consistent with a Gaussian ... we required that the x, y, xy, xx, and yy moments be strictly less than
 * 0.5, 0.5, 1.5, 36.5, and 36.5 respectively."  Reading R22: w = (I - min I) / sum(I - min I) (1/N for a constant
 * stamp); about the centre pixel, u, v in [-radius, radius] pixels:
 *     m_x = sum u w, m_y = sum v w, m_xy = sum u v w, m_xx = sum u^2 w, m_yy = sum v^2 w     (double precision)
 * keep = |m_x| < t[0] && |m_y| < t[1] && |m_xy| < t[2] && m_xx < t[3] && m_yy < t[4]; a stamp with a non-finite
 * pixel gets NaN moments and keep = 0.
 *   d_stamps      [n_stamps][2r+1][2r+1] float32 (e.g. kbmod_coadd_stamps' d_median)
 *   h_thresholds  [5] double on the HOST, or NULL for the paper's values
 *   d_moments     out [n_stamps][5] float64 (x, y, xy, xx, yy); may be NULL
 *   d_keep        out [n_stamps] uint8; may be NULL */
int kbmod_stamp_moments(const float* d_stamps, int n_stamps, int radius, const double* h_thresholds, double* d_moments,
                        uint8_t* d_keep, void* stream);

/* (a6) + the moment filter in one kernel (median stamp -> central moments): kbmod_coadd_stamps with
 * two more outputs computed from the median stamp while it is still on chip -- the same numbers, bit for bit, as
 * kbmod_stamp_moments(d_median).  d_mean, d_median, d_moments, d_keep may each be NULL. */
int kbmod_coadd_stamps_filtered(const float* d_img, const uint8_t* d_mask, int T, int H, int W, const double* h_times,
                                const int32_t* d_x0, const int32_t* d_y0, const float* d_vx, const float* d_vy,
                                const uint64_t* d_epoch_mask, int n_traj, int radius, float* d_mean, float* d_median,
                                const double* h_thresholds, double* d_moments, uint8_t* d_keep, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Whole path from HOST buffers (what bench.py's end-to-end number times): H2D copies of the
 * image / variance / mask stacks, kbmod_prepare_psi_phi, kbmod_search, D2H copies of the four
 * result arrays, then synchronises `stream`.  h_mask may be NULL.  Host buffers should be pinned
 * for the copies to run at full PCIe speed (pageable memory works, slower).
 *   d_arena  caller-owned device scratch of at least kbmod_pipeline_host_arena_bytes_for(...) bytes (exact for this
 *            velocity list; kbmod_pipeline_host_arena_bytes(...) is the upper bound for any list of n_vel entries) */
size_t kbmod_pipeline_host_arena_bytes(int T, int H, int W, int n_vel, const kbmod_search_params* p);
size_t kbmod_pipeline_host_arena_bytes_for(int T, int H, int W, const double* h_times, const float* h_vx, const float* h_vy,
                                           int n_vel, const kbmod_search_params* p);
int kbmod_pipeline_host(const float* h_img, const float* h_var, const uint8_t* h_mask, int T, int H, int W,
                        const float* h_psf, int n_psf, int k, const double* h_times, const float* h_vx,
                        const float* h_vy, int n_vel, const kbmod_search_params* p, float* h_lh, float* h_flux,
                        int32_t* h_vel_idx, int32_t* h_n_obs, void* d_arena, size_t arena_bytes, void* stream);

/* The same for n_stacks stacks of one shape searched with one grid (the 60 CCDs of a pointing group):
 * h_img[i], h_var[i], h_mask[i] (h_mask may be NULL) and the four result pointers per stack.  The copies of stack
 * i + 1 and of the results of stack i - 1 overlap the search of stack i (two internal copy streams, created once
 * per host thread and device, destroyed by kbmod_release_thread_state(); kernels run on `stream`; all stacks share one
 * plan).  d_arena: at least 2 x kbmod_pipeline_host_arena_bytes_for(...) bytes (1 x for a single stack).
 * Synchronises `stream` and both copy streams before returning, on success and on every error path. */
int kbmod_pipeline_host_batch(int n_stacks, const float* const* h_img, const float* const* h_var,
                              const uint8_t* const* h_mask, int T, int H, int W, const float* h_psf, int n_psf, int k,
                              const double* h_times, const float* h_vx, const float* h_vy, int n_vel,
                              const kbmod_search_params* p, float* const* h_lh, float* const* h_flux,
                              int32_t* const* h_vel_idx, int32_t* const* h_n_obs, void* d_arena, size_t arena_bytes,
                              void* stream);

/* Measurement helper for the roofline denominator (not part of the search path; synchronises): streams
 * conflict-free shared-memory loads of bytes_per_lane = 4, 8 or 16 on every SM and returns the best of three timed
 * repetitions in GB/s.  d_scratch4: 4 bytes of caller-owned device memory.  The theoretical figure is
 * SMs x 128 B/clk x SM clock. */
int kbmod_measure_smem_gbs(int bytes_per_lane, void* d_scratch4, double* h_gbs, void* stream);

/* Measurement helper: issue rate, in warp-instructions per SM clock per SM, of op = 0 FMNMX, 1 IADD3 (two register
 * operands), 2 FADD, 3 an alternative compare-exchange (FMNMX + three-register IADD3 recovering the maximum from the
 * bit patterns, plus one FADD that keeps the benchmark's chain alive).  On sm_100a FMNMX issues at 2 per clock per SM,
 * IADD3 and FADD at 4; the alternative exchange is no faster than two FMNMX.
 * Synchronises; d_scratch4 = 4 bytes of caller-owned device memory. */
int kbmod_measure_issue_rate(int op, void* d_scratch4, double* h_rate, void* stream);

const char* kbmod_last_error(void); /* thread-local, never NULL */
int kbmod_version(void);            /* 10000*major + 100*minor + patch */

#ifdef __cplusplus
}
#endif
#endif /* KBMOD_B200_H */
