// C-ABI entry points of libkbmod_b200.so (include/kbmod_b200.h): argument validation, host-side
// planning (displacement table, percentile ranks) and kernel launches.  No torch types, no
// device allocation, no CPU fallback.
#include <math.h>
#include <stdarg.h>
#include <string.h>

#include <vector>

#include "common.cuh"

// ---------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

void kb_set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char* kbmod_last_error(void) { return g_err; }
extern "C" int kbmod_version(void) { return 100; }

extern "C" void kbmod_default_params(kbmod_search_params* p) {
    if (!p) return;
    p->sigmag_enable = 1;
    p->pct_lo = 25.0f;
    p->pct_hi = 75.0f;
    p->sigmag_coeff = 0.7413f;
    p->n_sigma = 2.0f;
    p->filter_on = 0;
    p->min_lh = 10.0f;
    p->min_obs = 1;
    p->K = 8;
    p->algo = KBMOD_ALGO_AUTO;
}

// ---------------------------------------------------------------------------------------------
// phase timing: per host thread, off by default
struct PhaseMark { int phase; cudaEvent_t ev; };
static thread_local bool g_timing = false;
static thread_local std::vector<PhaseMark> g_marks;      // marks of the last kbmod_search
static thread_local std::vector<cudaEvent_t> g_pool;     // events to reuse

void kb_phase_mark(int phase, cudaStream_t st) {
    if (!g_timing) return;
    if (phase == KB_PHASE_START) {
        for (auto& m : g_marks) g_pool.push_back(m.ev);
        g_marks.clear();
    }
    cudaEvent_t ev = nullptr;
    if (!g_pool.empty()) { ev = g_pool.back(); g_pool.pop_back(); }
    else if (cudaEventCreate(&ev) != cudaSuccess) return;
    if (cudaEventRecord(ev, st) != cudaSuccess) { g_pool.push_back(ev); return; }
    g_marks.push_back({phase, ev});
}

extern "C" int kbmod_search_phase_timing(int enable) {
    g_timing = enable != 0;
    return KBMOD_OK;
}

extern "C" int kbmod_search_phase_ms(float* h_ms) {
    KB_REQUIRE(h_ms, KBMOD_ERR_INVALID_ARG, "NULL argument");
    for (int i = 0; i < 4; ++i) h_ms[i] = 0.0f;
    KB_REQUIRE(g_marks.size() >= 2, KBMOD_ERR_INVALID_ARG, "no timed kbmod_search on this thread (call kbmod_search_phase_timing(1) first)");
    KB_CUDA(cudaEventSynchronize(g_marks.back().ev));
    for (size_t i = 1; i < g_marks.size(); ++i) {
        float ms = 0.0f;
        KB_CUDA(cudaEventElapsedTime(&ms, g_marks[i - 1].ev, g_marks[i].ev));
        const int ph = g_marks[i].phase;
        if (ph >= 0 && ph < 4) h_ms[ph] += ms;
    }
    return KBMOD_OK;
}

static const int kSizes[] = {KB_SORTNET_SIZES};

int kb_padded_T(int T) {
    for (int s : kSizes)
        if (s >= T) return s;
    return -1;
}

// nearest-rank percentile index (reading R10): ceil(q n / 100) - 1 clamped to [0, n-1]
static int pct_rank(float q, int n) {
    int r = (int)ceil((double)q * (double)n / 100.0) - 1;
    if (r < 0) r = 0;
    if (r > n - 1) r = n - 1;
    return r;
}

int kb_make_dev_params(const kbmod_search_params* p, int T, DevParams* out) {
    KB_REQUIRE(p != nullptr, KBMOD_ERR_INVALID_ARG, "params is NULL");
    KB_REQUIRE(T >= 1, KBMOD_ERR_INVALID_ARG, "T = %d must be >= 1", T);
    KB_REQUIRE(T <= KBMOD_MAX_T, KBMOD_ERR_UNSUPPORTED, "T = %d exceeds %d", T, KBMOD_MAX_T);
    KB_REQUIRE(p->K >= 1, KBMOD_ERR_INVALID_ARG, "K = %d must be >= 1", p->K);
    KB_REQUIRE(p->K <= KBMOD_MAX_K, KBMOD_ERR_UNSUPPORTED, "K = %d exceeds %d", p->K, KBMOD_MAX_K);
    KB_REQUIRE(!(p->pct_lo < 0.0f) && !(p->pct_hi > 100.0f) && p->pct_lo <= p->pct_hi, KBMOD_ERR_INVALID_ARG,
               "percentiles (%g, %g) must satisfy 0 <= lo <= hi <= 100", p->pct_lo, p->pct_hi);
    KB_REQUIRE(!isnan(p->min_lh) && !isnan(p->n_sigma) && !isnan(p->sigmag_coeff), KBMOD_ERR_INVALID_ARG,
               "NaN parameter");
    KB_REQUIRE(p->algo >= KBMOD_ALGO_AUTO && p->algo <= KBMOD_ALGO_PRUNED, KBMOD_ERR_INVALID_ARG, "algo = %d",
               p->algo);
    memset(out, 0, sizeof(*out));
    out->sigmag_enable = p->sigmag_enable ? 1 : 0;
    out->filter_on = p->filter_on ? 1 : 0;
    out->min_obs = p->min_obs;
    out->K = p->K;
    out->T = T;
    out->coeff = p->sigmag_coeff;
    out->n_sigma = p->n_sigma;
    out->min_lh = p->min_lh;
    for (int n = 1; n <= KBMOD_MAX_T; ++n) {
        out->rk_lo[n] = (unsigned char)pct_rank(p->pct_lo, n);
        out->rk_md[n] = (unsigned char)pct_rank(50.0f, n);
        out->rk_hi[n] = (unsigned char)pct_rank(p->pct_hi, n);
    }
    return KBMOD_OK;
}

static int check_stack(int T, int H, int W) {
    KB_REQUIRE(T >= 1 && H >= 1 && W >= 1, KBMOD_ERR_INVALID_ARG, "T, H, W = %d, %d, %d must be >= 1", T, H, W);
    KB_REQUIRE(T <= KBMOD_MAX_T, KBMOD_ERR_UNSUPPORTED, "T = %d exceeds %d", T, KBMOD_MAX_T);
    KB_REQUIRE((double)T * H * W < 2147483648.0, KBMOD_ERR_UNSUPPORTED, "T*H*W = %.0f pixels exceeds 2^31",
               (double)T * H * W);
    return KBMOD_OK;
}

// reading R5: round half up; the multiply and the add are two separately rounded IEEE-double
// operations (the volatiles keep the host compiler from contracting them into one FMA)
static int32_t displacement(float v, double dt) {
    volatile double p = (double)v * dt;
    volatile double q = p + 0.5;
    return (int32_t)floor(q);
}

static void make_times(const double* h_times, int T, DevTimes* out) {
    memset(out, 0, sizeof(*out));
    for (int t = 0; t < T; ++t) out->dt[t] = h_times[t] - h_times[0];
}

extern "C" int kbmod_displacements(const double* h_times, int T, const float* h_vx, const float* h_vy, int n_vel,
                                   int32_t* h_dx, int32_t* h_dy) {
    KB_REQUIRE(h_times && h_vx && h_vy && h_dx && h_dy, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(T >= 1 && n_vel >= 0, KBMOD_ERR_INVALID_ARG, "T = %d, n_vel = %d", T, n_vel);
    for (int v = 0; v < n_vel; ++v)
        for (int t = 0; t < T; ++t) {
            const double dt = h_times[t] - h_times[0];
            h_dx[(size_t)v * T + t] = displacement(h_vx[v], dt);
            h_dy[(size_t)v * T + t] = displacement(h_vy[v], dt);
        }
    return KBMOD_OK;
}

// ---------------------------------------------------------------------------------------------
extern "C" int kbmod_prepare_psi_phi(const float* d_img, const float* d_var, const uint8_t* d_mask, int T, int H,
                                     int W, const float* h_psf, int n_psf, int k, float* d_psiphi, void* stream) {
    KB_REQUIRE(d_img && d_var && h_psf && d_psiphi, KBMOD_ERR_INVALID_ARG, "NULL argument");
    int rc = check_stack(T, H, W);
    if (rc) return rc;
    KB_REQUIRE(k >= 1 && (k & 1), KBMOD_ERR_INVALID_ARG, "PSF side k = %d must be odd and >= 1", k);
    KB_REQUIRE(k <= KBMOD_MAX_PSF, KBMOD_ERR_UNSUPPORTED, "PSF side k = %d exceeds %d", k, KBMOD_MAX_PSF);
    KB_REQUIRE(n_psf == 1 || n_psf == T, KBMOD_ERR_INVALID_ARG, "n_psf = %d must be 1 or T = %d", n_psf, T);
    return kb_launch_prep(d_img, d_var, d_mask, T, H, W, h_psf, n_psf, k, d_psiphi, (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------------------
// workspace layout of kbmod_search (all offsets 256-byte aligned)
struct SearchPlan {
    int TP;
    size_t off_stats, off_tab, off_pruned, pruned_bytes, total;
};

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static int plan_search(int T, int H, int W, int n_vel, const kbmod_search_params* p, SearchPlan* pl) {
    pl->TP = kb_padded_T(T);
    KB_REQUIRE(pl->TP > 0, KBMOD_ERR_UNSUPPORTED, "T = %d unsupported", T);
    size_t o = 0;
    pl->off_stats = o;
    o = align256(o + 8 * sizeof(unsigned long long));
    pl->off_tab = o;
    o = align256(o + (size_t)n_vel * pl->TP * sizeof(DispEntry));
    pl->off_pruned = o;
    // the pruned path's bound planes and key lists; not needed when the caller forces the direct kernel
    const int K = (p->K >= 1 && p->K <= KBMOD_MAX_K) ? p->K : 1;
    pl->pruned_bytes = (p->algo == KBMOD_ALGO_DIRECT) ? 0 : kb_pruned_workspace_bytes(T, H, W, n_vel, K);
    o = align256(o + pl->pruned_bytes);
    pl->total = o;
    return KBMOD_OK;
}

extern "C" size_t kbmod_search_workspace_bytes(int T, int H, int W, int n_vel, const kbmod_search_params* p) {
    SearchPlan pl;
    if (T < 1 || T > KBMOD_MAX_T || n_vel < 0 || !p) return 0;
    if (plan_search(T, H, W, n_vel, p, &pl)) return 0;
    return pl.total;
}

extern "C" int kbmod_search(const float* d_psiphi, int T, int H, int W, const double* h_times, const float* h_vx,
                            const float* h_vy, int n_vel, const kbmod_search_params* p, float* d_lh, float* d_flux,
                            int32_t* d_vel_idx, int32_t* d_n_obs, void* d_workspace, size_t workspace_bytes,
                            void* stream) {
    KB_REQUIRE(d_psiphi && h_times && d_lh && d_flux && d_vel_idx && d_n_obs && p, KBMOD_ERR_INVALID_ARG,
               "NULL argument");
    KB_REQUIRE(n_vel >= 0 && (n_vel == 0 || (h_vx && h_vy)), KBMOD_ERR_INVALID_ARG, "n_vel = %d / NULL velocities",
               n_vel);
    int rc = check_stack(T, H, W);
    if (rc) return rc;
    for (int t = 0; t < T; ++t) KB_REQUIRE(isfinite(h_times[t]), KBMOD_ERR_INVALID_ARG, "times[%d] is not finite", t);
    for (int v = 0; v < n_vel; ++v)
        KB_REQUIRE(isfinite(h_vx[v]) && isfinite(h_vy[v]), KBMOD_ERR_INVALID_ARG, "velocity %d is not finite", v);
    DevParams P;
    rc = kb_make_dev_params(p, T, &P);
    if (rc) return rc;
    SearchPlan pl;
    rc = plan_search(T, H, W, n_vel, p, &pl);
    if (rc) return rc;
    KB_REQUIRE(d_workspace && workspace_bytes >= pl.total, KBMOD_ERR_WORKSPACE,
               "workspace of %zu bytes is smaller than the %zu needed", workspace_bytes, pl.total);
    KB_REQUIRE(((uintptr_t)d_workspace & 255) == 0, KBMOD_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    char* ws = (char*)d_workspace;

    // (a2) displacement table, double precision on the host (reading R5)
    const int TP = pl.TP;
    const size_t plane = (size_t)H * W;
    std::vector<DispEntry> tab((size_t)n_vel * TP);
    std::vector<int32_t> hdx((size_t)n_vel * T), hdy((size_t)n_vel * T);
    KB_REQUIRE(W <= 32767 && H <= 32767, KBMOD_ERR_UNSUPPORTED, "W, H = %d, %d exceed 32767", W, H);
    for (int v = 0; v < n_vel; ++v)
        for (int t = 0; t < TP; ++t) {
            DispEntry e;
            if (t < T) {
                const double dt = h_times[t] - h_times[0];
                const int32_t dx = displacement(h_vx[v], dt), dy = displacement(h_vy[v], dt);
                hdx[(size_t)v * T + t] = dx;
                hdy[(size_t)v * T + t] = dy;
                // |d| beyond the image size can never land on-image: flag it so the entry fits int16 / int32
                const bool off_image = dx <= -W || dx >= W || dy <= -H || dy >= H;
                e.dx = off_image ? (int16_t)-32768 : (int16_t)dx;
                e.dy = off_image ? (int16_t)0 : (int16_t)dy;
                e.off = off_image ? 0 : (int32_t)((long long)t * (long long)plane + (long long)dy * W + dx);
            } else {
                e.dx = -32768;
                e.dy = 0;
                e.off = 0;
            }
            tab[(size_t)v * TP + t] = e;
        }

    // which kernel: the pruned one needs a finite threshold to prune against and a velocity list whose
    // groups can be staged
    int algo = p->algo;
    if (algo != KBMOD_ALGO_DIRECT && n_vel > 0) {
        double ps[4] = {0, 0, 0, 0};
        rc = kb_launch_search_pruned(nullptr, T, TP, H, W, nullptr, hdx.data(), hdy.data(), n_vel, p, P, nullptr, nullptr,
                                     nullptr, nullptr, nullptr, 0, nullptr, st, /*plan_only=*/1, ps, nullptr);
        if (algo == KBMOD_ALGO_AUTO) {
            const bool ok = rc == KBMOD_OK && isfinite(p->min_lh) && p->min_lh >= 3.0f && ps[0] <= 0.10 && ps[1] <= 4.0;
            algo = ok ? KBMOD_ALGO_PRUNED : KBMOD_ALGO_DIRECT;
        } else if (rc) {
            return rc;
        }
    } else {
        algo = KBMOD_ALGO_DIRECT;
    }
    unsigned long long stats[8] = {0, (unsigned long long)plane * n_vel, 1, (unsigned long long)algo, 0, 0, 0, 0};
    if (algo == KBMOD_ALGO_DIRECT) stats[0] = stats[1];
    // pageable source: cudaMemcpyAsync stages it before returning, so the vectors may go out of scope
    KB_CUDA(cudaMemcpyAsync(ws + pl.off_stats, stats, sizeof(stats), cudaMemcpyHostToDevice, st));
    if (n_vel > 0)
        KB_CUDA(cudaMemcpyAsync(ws + pl.off_tab, tab.data(), tab.size() * sizeof(DispEntry), cudaMemcpyHostToDevice,
                                st));
    const DispEntry* d_tab = (const DispEntry*)(ws + pl.off_tab);
    kb_phase_mark(KB_PHASE_START, st);
    if (algo == KBMOD_ALGO_DIRECT) {
        rc = kb_launch_search_direct(d_psiphi, T, TP, H, W, d_tab, n_vel, P, d_lh, d_flux, d_vel_idx, d_n_obs, st);
        kb_phase_mark(KB_PHASE_BOUND, st);  // the direct kernel is gather + filter + top-K in one: reported as phase 1
        return rc;
    }
    int launches = 0;
    rc = kb_launch_search_pruned(d_psiphi, T, TP, H, W, d_tab, hdx.data(), hdy.data(), n_vel, p, P, d_lh, d_flux,
                                 d_vel_idx, d_n_obs, ws + pl.off_pruned, pl.pruned_bytes,
                                 (unsigned long long*)(ws + pl.off_stats), st, 0, nullptr, &launches);
    if (rc) return rc;
    const unsigned long long nl = (unsigned long long)launches;  // kernels this call enqueued
    KB_CUDA(cudaMemcpyAsync(ws + pl.off_stats + 2 * sizeof(unsigned long long), &nl, sizeof(nl), cudaMemcpyHostToDevice, st));
    return KBMOD_OK;
}

// host-only view of the pruned search's plan (no GPU needed): what the planner would stage for this geometry
extern "C" int kbmod_plan_stats(int T, int H, int W, const double* h_times, const float* h_vx, const float* h_vy, int n_vel,
                                const kbmod_search_params* p, double* h_out) {
    KB_REQUIRE(h_times && h_out && p && (n_vel == 0 || (h_vx && h_vy)), KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n_vel >= 0, KBMOD_ERR_INVALID_ARG, "n_vel = %d", n_vel);
    int rc = check_stack(T, H, W);
    if (rc) return rc;
    DevParams P;
    rc = kb_make_dev_params(p, T, &P);
    if (rc) return rc;
    std::vector<int32_t> hdx((size_t)n_vel * T), hdy((size_t)n_vel * T);
    rc = kbmod_displacements(h_times, T, h_vx, h_vy, n_vel, hdx.data(), hdy.data());
    if (rc) return rc;
    double ps[4] = {0, 0, 0, 0};
    rc = kb_launch_search_pruned(nullptr, T, kb_padded_T(T), H, W, nullptr, hdx.data(), hdy.data(), n_vel, p, P, nullptr,
                                 nullptr, nullptr, nullptr, nullptr, 0, nullptr, nullptr, /*plan_only=*/1, ps, nullptr);
    if (rc) return rc;
    for (int i = 0; i < 4; ++i) h_out[i] = ps[i];
    return KBMOD_OK;
}

extern "C" int kbmod_search_stats(const void* d_workspace, unsigned long long* h_out) {
    KB_REQUIRE(d_workspace && h_out, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_CUDA(cudaMemcpy(h_out, d_workspace, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    return KBMOD_OK;
}

// ---------------------------------------------------------------------------------------------
extern "C" int kbmod_coadd_stamps(const float* d_img, const uint8_t* d_mask, int T, int H, int W,
                                  const double* h_times, const int32_t* d_x0, const int32_t* d_y0, const float* d_vx,
                                  const float* d_vy, const uint64_t* d_epoch_mask, int n_traj, int radius,
                                  float* d_mean, float* d_median, void* stream) {
    KB_REQUIRE(d_img && h_times, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n_traj >= 0, KBMOD_ERR_INVALID_ARG, "n_traj = %d", n_traj);
    int rc = check_stack(T, H, W);
    if (rc) return rc;
    KB_REQUIRE(radius >= 0, KBMOD_ERR_INVALID_ARG, "radius = %d", radius);
    KB_REQUIRE(radius <= KBMOD_MAX_STAMP_RADIUS, KBMOD_ERR_UNSUPPORTED, "radius = %d exceeds %d", radius,
               KBMOD_MAX_STAMP_RADIUS);
    if (n_traj == 0 || (!d_mean && !d_median)) return KBMOD_OK;
    KB_REQUIRE(d_x0 && d_y0 && d_vx && d_vy, KBMOD_ERR_INVALID_ARG, "NULL trajectory arrays");
    const int TP = kb_padded_T(T);
    DevTimes times;
    make_times(h_times, T, &times);
    return kb_launch_coadd(d_img, d_mask, T, TP, H, W, times, d_x0, d_y0, d_vx, d_vy,
                           (const unsigned long long*)d_epoch_mask, n_traj, radius, d_mean, d_median,
                           (cudaStream_t)stream);
}

extern "C" int kbmod_eval_trajectories(const float* d_psiphi, int T, int H, int W, const double* h_times,
                                       const int32_t* d_x0, const int32_t* d_y0, const float* d_vx,
                                       const float* d_vy, int n_traj, const kbmod_search_params* p, float* d_psi_lc,
                                       float* d_phi_lc, uint64_t* d_valid, uint64_t* d_kept, float* d_lh,
                                       float* d_flux, void* stream) {
    KB_REQUIRE(d_psiphi && h_times && p, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n_traj >= 0, KBMOD_ERR_INVALID_ARG, "n_traj = %d", n_traj);
    int rc = check_stack(T, H, W);
    if (rc) return rc;
    kbmod_search_params q = *p;
    if (q.K < 1 || q.K > KBMOD_MAX_K) q.K = 1;  // K is ignored here
    DevParams P;
    rc = kb_make_dev_params(&q, T, &P);
    if (rc) return rc;
    if (n_traj == 0) return KBMOD_OK;
    KB_REQUIRE(d_x0 && d_y0 && d_vx && d_vy, KBMOD_ERR_INVALID_ARG, "NULL trajectory arrays");
    DevTimes times;
    make_times(h_times, T, &times);
    return kb_launch_eval_trajectories(d_psiphi, T, kb_padded_T(T), H, W, times, d_x0, d_y0, d_vx, d_vy, n_traj, P,
                                       d_psi_lc, d_phi_lc, (unsigned long long*)d_valid, (unsigned long long*)d_kept,
                                       d_lh, d_flux, (cudaStream_t)stream);
}

extern "C" int kbmod_sigmag_filter(const float* d_psi_lc, const float* d_phi_lc, int n_lc, int T,
                                   const kbmod_search_params* p, uint64_t* d_kept, float* d_lh, float* d_flux,
                                   void* stream) {
    KB_REQUIRE(p, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n_lc >= 0, KBMOD_ERR_INVALID_ARG, "n_lc = %d", n_lc);
    kbmod_search_params q = *p;
    if (q.K < 1 || q.K > KBMOD_MAX_K) q.K = 1;
    DevParams P;
    int rc = kb_make_dev_params(&q, T, &P);
    if (rc) return rc;
    if (n_lc == 0) return KBMOD_OK;
    KB_REQUIRE(d_psi_lc && d_phi_lc, KBMOD_ERR_INVALID_ARG, "NULL lightcurves");
    return kb_launch_sigmag_filter(d_psi_lc, d_phi_lc, n_lc, T, kb_padded_T(T), P, (unsigned long long*)d_kept, d_lh,
                                   d_flux, (cudaStream_t)stream);
}

extern "C" int kbmod_stamp_moments(const float* d_stamps, int n_stamps, int radius, const double* h_thresholds,
                                   double* d_moments, uint8_t* d_keep, void* stream) {
    KB_REQUIRE(n_stamps >= 0, KBMOD_ERR_INVALID_ARG, "n_stamps = %d", n_stamps);
    KB_REQUIRE(radius >= 0, KBMOD_ERR_INVALID_ARG, "radius = %d", radius);
    KB_REQUIRE(radius <= KBMOD_MAX_STAMP_RADIUS, KBMOD_ERR_UNSUPPORTED, "radius = %d exceeds %d", radius,
               KBMOD_MAX_STAMP_RADIUS);
    if (n_stamps == 0 || (!d_moments && !d_keep)) return KBMOD_OK;
    KB_REQUIRE(d_stamps, KBMOD_ERR_INVALID_ARG, "NULL stamps");
    static const double paper[5] = {0.5, 0.5, 1.5, 36.5, 36.5};
    if (h_thresholds)
        for (int k = 0; k < 5; ++k) KB_REQUIRE(!isnan(h_thresholds[k]), KBMOD_ERR_INVALID_ARG, "NaN threshold");
    return kb_launch_stamp_moments(d_stamps, n_stamps, radius, h_thresholds ? h_thresholds : paper, d_moments, d_keep,
                                   (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------------------
// whole path from host buffers (bench.py's end-to-end number)
struct ArenaPlan {
    size_t off_img, off_var, off_mask, off_psiphi, off_lh, off_flux, off_vel, off_nobs, off_ws, ws_bytes, total;
};

static void plan_arena(int T, int H, int W, int n_vel, const kbmod_search_params* p, ArenaPlan* a) {
    const size_t px = (size_t)T * H * W, res = (size_t)H * W * p->K;
    size_t o = 0;
    a->off_img = o;    o = align256(o + px * 4);
    a->off_var = o;    o = align256(o + px * 4);
    a->off_mask = o;   o = align256(o + px);
    a->off_psiphi = o; o = align256(o + px * 8);
    a->off_lh = o;     o = align256(o + res * 4);
    a->off_flux = o;   o = align256(o + res * 4);
    a->off_vel = o;    o = align256(o + res * 4);
    a->off_nobs = o;   o = align256(o + res * 4);
    a->off_ws = o;
    a->ws_bytes = kbmod_search_workspace_bytes(T, H, W, n_vel, p);
    a->total = align256(o + a->ws_bytes);
}

extern "C" size_t kbmod_pipeline_host_arena_bytes(int T, int H, int W, int n_vel, const kbmod_search_params* p) {
    if (!p || T < 1 || T > KBMOD_MAX_T || H < 1 || W < 1 || n_vel < 0 || p->K < 1 || p->K > KBMOD_MAX_K) return 0;
    ArenaPlan a;
    plan_arena(T, H, W, n_vel, p, &a);
    return a.total;
}

extern "C" int kbmod_pipeline_host(const float* h_img, const float* h_var, const uint8_t* h_mask, int T, int H, int W,
                                   const float* h_psf, int n_psf, int k, const double* h_times, const float* h_vx,
                                   const float* h_vy, int n_vel, const kbmod_search_params* p, float* h_lh,
                                   float* h_flux, int32_t* h_vel_idx, int32_t* h_n_obs, void* d_arena,
                                   size_t arena_bytes, void* stream) {
    KB_REQUIRE(h_img && h_var && h_lh && h_flux && h_vel_idx && h_n_obs && p && d_arena, KBMOD_ERR_INVALID_ARG,
               "NULL argument");
    int rc = check_stack(T, H, W);
    if (rc) return rc;
    KB_REQUIRE(p->K >= 1 && p->K <= KBMOD_MAX_K, KBMOD_ERR_INVALID_ARG, "K = %d", p->K);
    KB_REQUIRE(((uintptr_t)d_arena & 255) == 0, KBMOD_ERR_INVALID_ARG, "arena must be 256-byte aligned");
    ArenaPlan a;
    plan_arena(T, H, W, n_vel, p, &a);
    KB_REQUIRE(arena_bytes >= a.total, KBMOD_ERR_WORKSPACE, "arena of %zu bytes is smaller than the %zu needed",
               arena_bytes, a.total);
    cudaStream_t st = (cudaStream_t)stream;
    char* A = (char*)d_arena;
    const size_t px = (size_t)T * H * W, res = (size_t)H * W * p->K;
    KB_CUDA(cudaMemcpyAsync(A + a.off_img, h_img, px * 4, cudaMemcpyHostToDevice, st));
    KB_CUDA(cudaMemcpyAsync(A + a.off_var, h_var, px * 4, cudaMemcpyHostToDevice, st));
    if (h_mask) KB_CUDA(cudaMemcpyAsync(A + a.off_mask, h_mask, px, cudaMemcpyHostToDevice, st));
    rc = kbmod_prepare_psi_phi((const float*)(A + a.off_img), (const float*)(A + a.off_var),
                               h_mask ? (const uint8_t*)(A + a.off_mask) : nullptr, T, H, W, h_psf, n_psf, k,
                               (float*)(A + a.off_psiphi), stream);
    if (rc) return rc;
    rc = kbmod_search((const float*)(A + a.off_psiphi), T, H, W, h_times, h_vx, h_vy, n_vel, p, (float*)(A + a.off_lh),
                      (float*)(A + a.off_flux), (int32_t*)(A + a.off_vel), (int32_t*)(A + a.off_nobs), A + a.off_ws,
                      a.ws_bytes, stream);
    if (rc) return rc;
    KB_CUDA(cudaMemcpyAsync(h_lh, A + a.off_lh, res * 4, cudaMemcpyDeviceToHost, st));
    KB_CUDA(cudaMemcpyAsync(h_flux, A + a.off_flux, res * 4, cudaMemcpyDeviceToHost, st));
    KB_CUDA(cudaMemcpyAsync(h_vel_idx, A + a.off_vel, res * 4, cudaMemcpyDeviceToHost, st));
    KB_CUDA(cudaMemcpyAsync(h_n_obs, A + a.off_nobs, res * 4, cudaMemcpyDeviceToHost, st));
    KB_CUDA(cudaStreamSynchronize(st));
    return KBMOD_OK;
}

// ---------------------------------------------------------------------------------------------
// a batch of stacks of one shape (the CCDs of a pointing group): copies overlap the searches
struct BatchStreams {
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t in_done[2] = {nullptr, nullptr}, comp_done[2] = {nullptr, nullptr}, out_done[2] = {nullptr, nullptr};
    bool ready = false;
};
static thread_local BatchStreams g_bs;

extern "C" int kbmod_pipeline_host_batch(int n_stacks, const float* const* h_img, const float* const* h_var,
                                         const uint8_t* const* h_mask, int T, int H, int W, const float* h_psf, int n_psf,
                                         int k, const double* h_times, const float* h_vx, const float* h_vy, int n_vel,
                                         const kbmod_search_params* p, float* const* h_lh, float* const* h_flux,
                                         int32_t* const* h_vel_idx, int32_t* const* h_n_obs, void* d_arena,
                                         size_t arena_bytes, void* stream) {
    KB_REQUIRE(n_stacks >= 0, KBMOD_ERR_INVALID_ARG, "n_stacks = %d", n_stacks);
    if (n_stacks == 0) return KBMOD_OK;
    KB_REQUIRE(h_img && h_var && h_lh && h_flux && h_vel_idx && h_n_obs && p && d_arena, KBMOD_ERR_INVALID_ARG, "NULL argument");
    int rc = check_stack(T, H, W);
    if (rc) return rc;
    KB_REQUIRE(p->K >= 1 && p->K <= KBMOD_MAX_K, KBMOD_ERR_INVALID_ARG, "K = %d", p->K);
    KB_REQUIRE(((uintptr_t)d_arena & 255) == 0, KBMOD_ERR_INVALID_ARG, "arena must be 256-byte aligned");
    ArenaPlan a;
    plan_arena(T, H, W, n_vel, p, &a);
    const int n_buf = n_stacks > 1 ? 2 : 1;
    KB_REQUIRE(arena_bytes >= (size_t)n_buf * a.total, KBMOD_ERR_WORKSPACE,
               "arena of %zu bytes is smaller than the %d x %zu needed", arena_bytes, n_buf, a.total);
    for (int i = 0; i < n_stacks; ++i)
        KB_REQUIRE(h_img[i] && h_var[i] && h_lh[i] && h_flux[i] && h_vel_idx[i] && h_n_obs[i], KBMOD_ERR_INVALID_ARG,
                   "NULL buffer of stack %d", i);
    if (!g_bs.ready) {
        KB_CUDA(cudaStreamCreateWithFlags(&g_bs.s_in, cudaStreamNonBlocking));
        KB_CUDA(cudaStreamCreateWithFlags(&g_bs.s_out, cudaStreamNonBlocking));
        for (int b = 0; b < 2; ++b) {
            KB_CUDA(cudaEventCreateWithFlags(&g_bs.in_done[b], cudaEventDisableTiming));
            KB_CUDA(cudaEventCreateWithFlags(&g_bs.comp_done[b], cudaEventDisableTiming));
            KB_CUDA(cudaEventCreateWithFlags(&g_bs.out_done[b], cudaEventDisableTiming));
        }
        g_bs.ready = true;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t px = (size_t)T * H * W, res = (size_t)H * W * p->K;
    // everything enqueued on `stream` before this call happens-before the first copy
    KB_CUDA(cudaEventRecord(g_bs.comp_done[1], st));
    KB_CUDA(cudaStreamWaitEvent(g_bs.s_in, g_bs.comp_done[1], 0));
    for (int i = 0; i < n_stacks; ++i) {
        const int b = i & 1;
        char* A = (char*)d_arena + (size_t)b * a.total;
        const uint8_t* hm = h_mask ? h_mask[i] : nullptr;
        // inputs of buffer b are free once the search of stack i - 2 is done
        if (i >= 2) KB_CUDA(cudaStreamWaitEvent(g_bs.s_in, g_bs.comp_done[b], 0));
        KB_CUDA(cudaMemcpyAsync(A + a.off_img, h_img[i], px * 4, cudaMemcpyHostToDevice, g_bs.s_in));
        KB_CUDA(cudaMemcpyAsync(A + a.off_var, h_var[i], px * 4, cudaMemcpyHostToDevice, g_bs.s_in));
        if (hm) KB_CUDA(cudaMemcpyAsync(A + a.off_mask, hm, px, cudaMemcpyHostToDevice, g_bs.s_in));
        KB_CUDA(cudaEventRecord(g_bs.in_done[b], g_bs.s_in));
        // the search waits for its inputs and for the results of stack i - 2 to have left buffer b
        KB_CUDA(cudaStreamWaitEvent(st, g_bs.in_done[b], 0));
        if (i >= 2) KB_CUDA(cudaStreamWaitEvent(st, g_bs.out_done[b], 0));
        rc = kbmod_prepare_psi_phi((const float*)(A + a.off_img), (const float*)(A + a.off_var),
                                   hm ? (const uint8_t*)(A + a.off_mask) : nullptr, T, H, W, h_psf, n_psf, k,
                                   (float*)(A + a.off_psiphi), stream);
        if (rc) return rc;
        rc = kbmod_search((const float*)(A + a.off_psiphi), T, H, W, h_times, h_vx, h_vy, n_vel, p, (float*)(A + a.off_lh),
                          (float*)(A + a.off_flux), (int32_t*)(A + a.off_vel), (int32_t*)(A + a.off_nobs), A + a.off_ws,
                          a.ws_bytes, stream);
        if (rc) return rc;
        KB_CUDA(cudaEventRecord(g_bs.comp_done[b], st));
        KB_CUDA(cudaStreamWaitEvent(g_bs.s_out, g_bs.comp_done[b], 0));
        KB_CUDA(cudaMemcpyAsync(h_lh[i], A + a.off_lh, res * 4, cudaMemcpyDeviceToHost, g_bs.s_out));
        KB_CUDA(cudaMemcpyAsync(h_flux[i], A + a.off_flux, res * 4, cudaMemcpyDeviceToHost, g_bs.s_out));
        KB_CUDA(cudaMemcpyAsync(h_vel_idx[i], A + a.off_vel, res * 4, cudaMemcpyDeviceToHost, g_bs.s_out));
        KB_CUDA(cudaMemcpyAsync(h_n_obs[i], A + a.off_nobs, res * 4, cudaMemcpyDeviceToHost, g_bs.s_out));
        KB_CUDA(cudaEventRecord(g_bs.out_done[b], g_bs.s_out));
    }
    // the caller's stream finishes after the last result has landed
    KB_CUDA(cudaStreamWaitEvent(st, g_bs.out_done[(n_stacks - 1) & 1], 0));
    if (n_stacks > 1) KB_CUDA(cudaStreamWaitEvent(st, g_bs.out_done[(n_stacks - 2) & 1], 0));
    KB_CUDA(cudaStreamSynchronize(st));
    return KBMOD_OK;
}
