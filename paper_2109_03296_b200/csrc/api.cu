// C-ABI entry points of libkbmod_b200.so (include/kbmod_b200.h): argument validation, host-side
// planning (displacement table, percentile ranks) and kernel launches.  No torch types, no
// device allocation, no CPU fallback.
#include <math.h>
#include <stdarg.h>
#include <string.h>

#include <algorithm>
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
    p->pct_interp = 0;
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
    out->pct_interp = p->pct_interp ? 1 : 0;
    const float qs[3] = {p->pct_lo, 50.0f, p->pct_hi};
    unsigned char* rk[3] = {out->rk_lo, out->rk_md, out->rk_hi};
    float* fr[3] = {out->fr_lo, out->fr_md, out->fr_hi};
    for (int i = 0; i < 3; ++i) {
        rk[i][0] = 0;
        fr[i][0] = -1.0f;
        for (int n = 1; n <= KBMOD_MAX_T; ++n) {
            if (!out->pct_interp) {
                rk[i][n] = (unsigned char)pct_rank(qs[i], n);
                fr[i][n] = -1.0f;
                continue;
            }
            // reading R23: position h = (n - 1) q / 100 in the ascending sort, linear between its neighbours
            const double h = (double)(n - 1) * (double)qs[i] / 100.0;
            if (h <= 0.0) { rk[i][n] = 0; fr[i][n] = -1.0f; }
            else if (h >= (double)(n - 1)) { rk[i][n] = (unsigned char)(n - 1); fr[i][n] = -1.0f; }
            else {
                const int k = (int)floor(h);
                rk[i][n] = (unsigned char)k;
                fr[i][n] = (float)(h - (double)k);
            }
        }
    }
    return KBMOD_OK;
}

// host-only: the percentile positions the kernels use for n valid samples (what the -m "not gpu" tests pin against
// the oracle for user percentiles such as 10 / 90)
extern "C" int kbmod_percentile_ranks(const kbmod_search_params* p, int n, int* h_k, float* h_g) {
    KB_REQUIRE(p && h_k && h_g, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n >= 1 && n <= KBMOD_MAX_T, KBMOD_ERR_INVALID_ARG, "n = %d must be in [1, %d]", n, KBMOD_MAX_T);
    kbmod_search_params q = *p;
    if (q.K < 1 || q.K > KBMOD_MAX_K) q.K = 1;
    DevParams P;
    const int rc = kb_make_dev_params(&q, n, &P);
    if (rc) return rc;
    h_k[0] = P.rk_lo[n]; h_k[1] = P.rk_md[n]; h_k[2] = P.rk_hi[n];
    h_g[0] = P.fr_lo[n]; h_g[1] = P.fr_md[n]; h_g[2] = P.fr_hi[n];
    return KBMOD_OK;
}

static int check_stack(int T, int H, int W) {
    KB_REQUIRE(T >= 1 && H >= 1 && W >= 1, KBMOD_ERR_INVALID_ARG, "T, H, W = %d, %d, %d must be >= 1", T, H, W);
    KB_REQUIRE(T <= KBMOD_MAX_T, KBMOD_ERR_UNSUPPORTED, "T = %d exceeds %d", T, KBMOD_MAX_T);
    KB_REQUIRE((double)T * H * W < 2147483648.0, KBMOD_ERR_UNSUPPORTED, "T*H*W = %.0f pixels exceeds 2^31",
               (double)T * H * W);
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
// The search plan: everything kbmod_search derives from the geometry alone (T, H, W, the row band, epoch times,
// the velocity list, the parameters) -- the displacement table (a2), the S4 canvas geometry and offset table, the
// choice of kernel, the pruned kernel's velocity groups / staging geometry / on-image masks -- packed into ONE
// host blob (pinned when a CUDA context exists) that a search uploads with a single asynchronous copy, plus the
// workspace layout.  Immutable after creation: any number of searches, on any streams, may share one plan, each
// with its own workspace.
struct kbmod_plan {
    int T = 0, TP = 0, H = 0, W = 0, row_begin = 0, row_end = 0, n_vel = 0, algo = 0, device = -1;
    kbmod_search_params p{};
    DevParams P{};
    std::vector<double> times;
    std::vector<float> vx, vy;
    S4Geom G{};
    PrunedPlan pr;
    bool has_pruned = false;
    // host blob of the device tables and where each table sits in it
    unsigned char* blob = nullptr;
    bool blob_pinned = false;
    size_t blob_bytes = 0, b_off = 0, b_order = 0, b_gvel = 0, b_gtbl = 0, b_maskx = 0, b_masky = 0, b_gfoot = 0;
    // workspace layout (all offsets 256-byte aligned)
    size_t w_stats = 0, w_tables = 0, w_keys = 0, w_s4 = 0, w_scratch = 0, scratch_bytes = 0, w_total = 0;
    cudaEvent_t uploaded = nullptr;  // recorded after the last upload from the blob: the blob may be freed after it
};

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

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

extern "C" void kbmod_plan_destroy(kbmod_plan* pl) {
    if (!pl) return;
    if (pl->uploaded) {
        cudaEventSynchronize(pl->uploaded);  // an upload from the blob may still be in flight
        cudaEventDestroy(pl->uploaded);
    }
    if (pl->blob) {
        if (pl->blob_pinned) cudaFreeHost(pl->blob);
        else free(pl->blob);
    }
    delete pl;
}

extern "C" int kbmod_plan_create(int T, int H, int W, const double* h_times, const float* h_vx, const float* h_vy,
                                 int n_vel, const kbmod_search_params* p, int row_begin, int row_end,
                                 kbmod_plan** out) {
    KB_REQUIRE(out, KBMOD_ERR_INVALID_ARG, "NULL argument");
    *out = nullptr;
    KB_REQUIRE(h_times && p, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n_vel >= 0 && (n_vel == 0 || (h_vx && h_vy)), KBMOD_ERR_INVALID_ARG, "n_vel = %d / NULL velocities", n_vel);
    int rc = check_stack(T, H, W);
    if (rc) return rc;
    KB_REQUIRE(W <= 32767 && H <= 32767, KBMOD_ERR_UNSUPPORTED, "W, H = %d, %d exceed 32767", W, H);
    KB_REQUIRE(row_begin >= 0 && row_begin <= row_end && row_end <= H, KBMOD_ERR_INVALID_ARG,
               "row band [%d, %d) must lie inside [0, %d]", row_begin, row_end, H);
    for (int t = 0; t < T; ++t) KB_REQUIRE(isfinite(h_times[t]), KBMOD_ERR_INVALID_ARG, "times[%d] is not finite", t);
    for (int v = 0; v < n_vel; ++v)
        KB_REQUIRE(isfinite(h_vx[v]) && isfinite(h_vy[v]), KBMOD_ERR_INVALID_ARG, "velocity %d is not finite", v);
    kbmod_plan* pl = new kbmod_plan();
    struct Guard { kbmod_plan* p; ~Guard() { if (p) kbmod_plan_destroy(p); } } guard{pl};
    rc = kb_make_dev_params(p, T, &pl->P);
    if (rc) return rc;
    pl->T = T; pl->H = H; pl->W = W; pl->row_begin = row_begin; pl->row_end = row_end; pl->n_vel = n_vel;
    pl->p = *p;
    pl->TP = kb_padded_T(T);
    KB_REQUIRE(pl->TP > 0, KBMOD_ERR_UNSUPPORTED, "T = %d unsupported", T);
    pl->times.assign(h_times, h_times + T);
    if (n_vel) { pl->vx.assign(h_vx, h_vx + n_vel); pl->vy.assign(h_vy, h_vy + n_vel); }

    // (a2) displacement table, double precision on the host (reading R5)
    std::vector<int32_t> hdx((size_t)n_vel * T), hdy((size_t)n_vel * T);
    if (n_vel) {
        rc = kbmod_displacements(h_times, T, h_vx, h_vy, n_vel, hdx.data(), hdy.data());
        if (rc) return rc;
    }
    std::vector<int32_t> off;
    rc = kb_s4_plan(T, pl->TP, H, W, hdx.data(), hdy.data(), n_vel, &pl->G, &off);
    if (rc) return rc;

    // which kernel: the pruned one needs a finite threshold to prune against and a velocity list whose groups can
    // be staged
    int algo = p->algo;
    const int n_rows = row_end - row_begin;
    if (algo != KBMOD_ALGO_DIRECT && n_vel > 0 && n_rows > 0) {
        rc = kb_pruned_plan_build(T, H, W, row_begin, row_end, hdx.data(), hdy.data(), n_vel, &pl->pr);
        const double per_eval = pl->pr.evals > 0 ? pl->pr.staged / pl->pr.evals : 0.0;
        if (algo == KBMOD_ALGO_AUTO) {
            const bool ok = rc == KBMOD_OK && isfinite(p->min_lh) && p->min_lh >= 3.0f && !pl->pr.too_scattered && per_eval <= 4.0;
            algo = ok ? KBMOD_ALGO_PRUNED : KBMOD_ALGO_DIRECT;
        } else {
            if (rc) return rc;
            KB_REQUIRE(!pl->pr.too_scattered, KBMOD_ERR_UNSUPPORTED,
                       "pruned search: %d velocity groups (velocities too scattered; use the direct kernel)", pl->pr.ng);
        }
        pl->has_pruned = algo == KBMOD_ALGO_PRUNED;
    } else {
        algo = KBMOD_ALGO_DIRECT;
    }
    pl->algo = algo;
    if (!pl->has_pruned) pl->pr = PrunedPlan();

    // the order in which the direct kernel walks the velocities: neighbours in the list are neighbours in
    // displacement space (bands of a few rows of the displacement at the epoch farthest from times[0], swept in x in
    // alternating directions), so consecutive velocities of a warp touch overlapping cache lines.  Results do not
    // depend on it (the top-K keys carry the velocity index).
    std::vector<int32_t> order(n_vel);
    {
        int t_far = 0;
        double best = -1.0;
        for (int t = 0; t < T; ++t)
            if (fabs(h_times[t] - h_times[0]) > best) { best = fabs(h_times[t] - h_times[0]); t_far = t; }
        const int band = 6;
        for (int v = 0; v < n_vel; ++v) order[v] = v;
        auto key = [&](int v) {
            const long long dx = hdx[(size_t)v * T + t_far], dy = hdy[(size_t)v * T + t_far];
            const long long b = (dy >= 0 ? dy : dy - (band - 1)) / band;
            return std::make_pair(b, (b & 1) ? -dx : dx);
        };
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return key(a) < key(b); });
    }

    // ---- the blob
    size_t o = 0;
    pl->b_off = o;   o = align256(o + off.size() * 4);
    pl->b_order = o; o = align256(o + order.size() * 4);
    pl->b_gvel = o;  o = align256(o + pl->pr.gvel.size() * 4);
    pl->b_gtbl = o;  o = align256(o + pl->pr.gtbl.size());
    pl->b_maskx = o; o = align256(o + pl->pr.maskx.size() * 8);
    pl->b_masky = o; o = align256(o + pl->pr.masky.size() * 8);
    pl->b_gfoot = o; o = align256(o + pl->pr.gfoot.size() * 4);
    pl->blob_bytes = std::max<size_t>(o, 256);
    void* hp = nullptr;
    if (cudaMallocHost(&hp, pl->blob_bytes) == cudaSuccess) {
        pl->blob = (unsigned char*)hp;
        pl->blob_pinned = true;
        cudaGetDevice(&pl->device);
    } else {
        cudaGetLastError();  // no CUDA context (host-only use, e.g. kbmod_plan_stats): pageable memory will do
        pl->blob = (unsigned char*)malloc(pl->blob_bytes);
        KB_REQUIRE(pl->blob, KBMOD_ERR_INVALID_ARG, "out of host memory");
    }
    memset(pl->blob, 0, pl->blob_bytes);
    if (!off.empty()) memcpy(pl->blob + pl->b_off, off.data(), off.size() * 4);
    if (!order.empty()) memcpy(pl->blob + pl->b_order, order.data(), order.size() * 4);
    if (pl->has_pruned) {
        memcpy(pl->blob + pl->b_gvel, pl->pr.gvel.data(), pl->pr.gvel.size() * 4);
        memcpy(pl->blob + pl->b_gtbl, pl->pr.gtbl.data(), pl->pr.gtbl.size());
        memcpy(pl->blob + pl->b_maskx, pl->pr.maskx.data(), pl->pr.maskx.size() * 8);
        memcpy(pl->blob + pl->b_masky, pl->pr.masky.data(), pl->pr.masky.size() * 8);
        memcpy(pl->blob + pl->b_gfoot, pl->pr.gfoot.data(), pl->pr.gfoot.size() * 4);
        // the device copies are what the kernels read; the host vectors are no longer needed
        std::vector<int32_t>().swap(pl->pr.gvel);
        std::vector<unsigned char>().swap(pl->pr.gtbl);
        std::vector<unsigned long long>().swap(pl->pr.maskx);
        std::vector<unsigned long long>().swap(pl->pr.masky);
        std::vector<uint32_t>().swap(pl->pr.gfoot);
    }

    // ---- workspace layout
    o = 0;
    pl->w_stats = o;  o = align256(o + 8 * sizeof(unsigned long long));
    pl->w_tables = o; o = align256(o + pl->blob_bytes);
    pl->w_keys = o;   o = align256(o + (size_t)n_rows * W * pl->P.K * 8);
    pl->w_s4 = o;     o = align256(o + kb_s4_bytes(pl->G, T));
    pl->w_scratch = o;
    pl->scratch_bytes = pl->has_pruned ? kb_pruned_scratch_bytes(T, H, W, n_rows, n_vel) : 0;
    o = align256(o + pl->scratch_bytes);
    pl->w_total = o;
    guard.p = nullptr;
    *out = pl;
    return KBMOD_OK;
}

extern "C" size_t kbmod_plan_workspace_bytes(const kbmod_plan* pl) { return pl ? pl->w_total : 0; }

extern "C" int kbmod_plan_info(const kbmod_plan* pl, double* h_out) {
    KB_REQUIRE(pl && h_out, KBMOD_ERR_INVALID_ARG, "NULL argument");
    h_out[0] = (double)pl->algo;
    h_out[1] = (double)pl->pr.ng;
    h_out[2] = pl->pr.evals > 0 ? pl->pr.staged / pl->pr.evals : 0.0;
    h_out[3] = pl->pr.off_image;
    h_out[4] = (double)pl->G.Wp;
    h_out[5] = (double)pl->G.Hp;
    h_out[6] = (double)pl->pr.too_scattered;
    h_out[7] = (double)pl->blob_bytes;
    h_out[8] = pl->pr.gather_fraction;
    h_out[9] = (double)pl->w_total;
    return KBMOD_OK;
}

// the plan's tables -> the workspace (one asynchronous copy from the pinned blob; no host synchronisation)
static int plan_upload_tables(kbmod_plan* pl, void* d_workspace, cudaStream_t st) {
    if (!pl->uploaded) KB_CUDA(cudaEventCreateWithFlags(&pl->uploaded, cudaEventDisableTiming));
    KB_CUDA(cudaMemcpyAsync((char*)d_workspace + pl->w_tables, pl->blob, pl->blob_bytes, cudaMemcpyHostToDevice, st));
    KB_CUDA(cudaEventRecord(pl->uploaded, st));
    return KBMOD_OK;
}

static int plan_search_impl(kbmod_plan* pl, const float* d_psiphi, float* d_lh, float* d_flux, int32_t* d_vel_idx,
                            int32_t* d_n_obs, void* d_workspace, size_t workspace_bytes, void* stream, bool upload_tables);

extern "C" int kbmod_plan_search(kbmod_plan* pl, const float* d_psiphi, float* d_lh, float* d_flux, int32_t* d_vel_idx,
                                 int32_t* d_n_obs, void* d_workspace, size_t workspace_bytes, void* stream) {
    return plan_search_impl(pl, d_psiphi, d_lh, d_flux, d_vel_idx, d_n_obs, d_workspace, workspace_bytes, stream, true);
}

// upload_tables = false: the caller has put the plan's tables into this workspace already and nothing has written
// there since (kbmod_pipeline_host_batch does, once per arena half: a table upload behind every search would queue
// on the host-to-device copy engine after the next stack's 2 GB of inputs and hold the search up for their 35 ms)
static int plan_search_impl(kbmod_plan* pl, const float* d_psiphi, float* d_lh, float* d_flux, int32_t* d_vel_idx,
                            int32_t* d_n_obs, void* d_workspace, size_t workspace_bytes, void* stream, bool upload_tables) {
    KB_REQUIRE(pl && d_psiphi, KBMOD_ERR_INVALID_ARG, "NULL argument");
    if (pl->row_end == pl->row_begin) return KBMOD_OK;  // an empty band: nothing to search, nothing to write
    KB_REQUIRE(d_lh && d_flux && d_vel_idx && d_n_obs, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(d_workspace && workspace_bytes >= pl->w_total, KBMOD_ERR_WORKSPACE,
               "workspace of %zu bytes is smaller than the %zu needed", workspace_bytes, pl->w_total);
    KB_REQUIRE(((uintptr_t)d_workspace & 255) == 0, KBMOD_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    char* ws = (char*)d_workspace;
    const int n_rows = pl->row_end - pl->row_begin;
    const unsigned long long plane = (unsigned long long)n_rows * pl->W;
    unsigned long long* d_stats = (unsigned long long*)(ws + pl->w_stats);
    unsigned long long* d_keys = (unsigned long long*)(ws + pl->w_keys);
    void* d_S4 = ws + pl->w_s4;
    const int* d_off = (const int*)(ws + pl->w_tables + pl->b_off);

    // stats + tables: one copy from the plan's blob (pinned: asynchronous, no host synchronisation); the 64 stats
    // bytes ride in front of the tables
    if (upload_tables) {
        const int rcu = plan_upload_tables(pl, d_workspace, st);
        if (rcu) return rcu;
    }
    unsigned long long stats[8] = {0, plane * (unsigned long long)pl->n_vel, 2, (unsigned long long)pl->algo, 0, 0, 0, 0};
    if (pl->algo == KBMOD_ALGO_DIRECT) stats[0] = stats[1];
    KB_CUDA(cudaMemsetAsync(d_stats, 0, 8 * sizeof(unsigned long long), st));
    kb_phase_mark(KB_PHASE_START, st);
    int rc = kb_launch_s4_build(d_psiphi, pl->T, pl->H, pl->W, pl->G, pl->P.filter_on, d_S4, st);
    if (rc) return rc;
    int launches = 2;  // s4_build + finalize
    if (pl->algo == KBMOD_ALGO_DIRECT) {
        kb_phase_mark(KB_PHASE_PLANES, st);
        rc = kb_launch_search_direct(pl->TP, d_S4, pl->G, d_off, (const int*)(ws + pl->w_tables + pl->b_order), pl->W,
                                     pl->row_begin, pl->row_end, pl->n_vel, pl->P, d_keys, d_stats + 7 /* work counter */, st);
        if (rc) return rc;
        if (n_rows > 0) ++launches;
        kb_phase_mark(KB_PHASE_BOUND, st);  // the direct kernel is gather + filter + top-K in one: reported as phase 1
    } else {
        PrunedTablesDev tb;
        char* tbl = ws + pl->w_tables;
        tb.gvel = (const int32_t*)(tbl + pl->b_gvel);
        tb.gtbl = (const unsigned char*)(tbl + pl->b_gtbl);
        tb.maskx = (const unsigned long long*)(tbl + pl->b_maskx);
        tb.masky = (const unsigned long long*)(tbl + pl->b_masky);
        tb.gfoot = (const uint32_t*)(tbl + pl->b_gfoot);
        int nl = 0;
        rc = kb_launch_search_pruned(d_psiphi, pl->pr, tb, pl->TP, d_S4, pl->G, d_off, &pl->p, pl->P, d_keys, ws + pl->w_scratch,
                                     pl->scratch_bytes, d_stats, st, &nl);
        if (rc) return rc;
        launches += nl;
    }
    rc = kb_launch_finalize(pl->TP, d_keys, d_S4, pl->G, d_off, pl->W, pl->row_begin, n_rows, pl->P, d_lh, d_flux, d_vel_idx,
                            d_n_obs, st);
    if (rc) return rc;
    kb_phase_mark(KB_PHASE_FINALIZE, st);
    // [1] nominal count, [2] kernels launched, [3] kernel used ([0], trajectories fully evaluated, is counted by the
    // exact kernels of the pruned path on the device; the direct kernel evaluates them all)
    stats[2] = (unsigned long long)launches + 1;  // + the one-thread kernel that writes these counters
    return kb_write_stats(d_stats, stats[1], stats[2], stats[3], pl->algo == KBMOD_ALGO_DIRECT ? stats[1] : 0ull, st);
}

// unfiltered sum-LH of the result slots of the last kbmod_plan_search that used this workspace
extern "C" int kbmod_plan_unfiltered_lh(const kbmod_plan* pl, const void* d_workspace, const int32_t* d_vel_idx,
                                        float* d_lh_raw, void* stream) {
    KB_REQUIRE(pl && d_workspace && d_vel_idx && d_lh_raw, KBMOD_ERR_INVALID_ARG, "NULL argument");
    const char* ws = (const char*)d_workspace;
    return kb_launch_unfiltered_lh(pl->TP, d_vel_idx, ws + pl->w_s4, pl->G, (const int*)(ws + pl->w_tables + pl->b_off),
                                   pl->W, pl->row_begin, pl->row_end - pl->row_begin, pl->P.K, pl->n_vel, pl->P.filter_on, d_lh_raw,
                                   (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------------------
// kbmod_search: the one-call form.  It keeps ONE plan per host thread and rebuilds it when the geometry changes
// (searching the 60 CCDs of a pointing group with one grid reuses it); kbmod_release_thread_state() frees it.
static thread_local kbmod_plan* g_plan = nullptr;

static bool plan_matches(const kbmod_plan* pl, int T, int H, int W, const double* h_times, const float* h_vx,
                         const float* h_vy, int n_vel, const kbmod_search_params* p, int row_begin, int row_end) {
    if (!pl || pl->T != T || pl->H != H || pl->W != W || pl->n_vel != n_vel || pl->row_begin != row_begin ||
        pl->row_end != row_end || memcmp(&pl->p, p, sizeof(*p)) != 0)
        return false;
    int dev = -1;
    if (pl->blob_pinned && (cudaGetDevice(&dev) != cudaSuccess || dev != pl->device)) return false;
    if (memcmp(pl->times.data(), h_times, (size_t)T * sizeof(double)) != 0) return false;
    if (n_vel && (memcmp(pl->vx.data(), h_vx, (size_t)n_vel * 4) != 0 || memcmp(pl->vy.data(), h_vy, (size_t)n_vel * 4) != 0))
        return false;
    return true;
}

static int thread_plan(int T, int H, int W, const double* h_times, const float* h_vx, const float* h_vy, int n_vel,
                       const kbmod_search_params* p, int row_begin, int row_end, kbmod_plan** out) {
    KB_REQUIRE(h_times && p && (n_vel == 0 || (h_vx && h_vy)), KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n_vel >= 0, KBMOD_ERR_INVALID_ARG, "n_vel = %d", n_vel);
    if (T >= 1 && T <= KBMOD_MAX_T && plan_matches(g_plan, T, H, W, h_times, h_vx, h_vy, n_vel, p, row_begin, row_end)) {
        *out = g_plan;
        return KBMOD_OK;
    }
    kbmod_plan* np = nullptr;
    int rc = kbmod_plan_create(T, H, W, h_times, h_vx, h_vy, n_vel, p, row_begin, row_end, &np);
    if (rc) return rc;
    kbmod_plan_destroy(g_plan);
    g_plan = np;
    *out = np;
    return KBMOD_OK;
}

extern "C" size_t kbmod_search_workspace_bytes_for(int T, int H, int W, const double* h_times, const float* h_vx,
                                                   const float* h_vy, int n_vel, const kbmod_search_params* p,
                                                   int row_begin, int row_end) {
    kbmod_plan* pl = nullptr;
    if (thread_plan(T, H, W, h_times, h_vx, h_vy, n_vel, p, row_begin, row_end, &pl)) return 0;
    return pl->w_total;
}

// upper bound for any velocity list of n_vel entries: the canvas padded by the whole image on every side
extern "C" size_t kbmod_search_workspace_bytes(int T, int H, int W, int n_vel, const kbmod_search_params* p) {
    if (T < 1 || T > KBMOD_MAX_T || H < 1 || W < 1 || n_vel < 0 || !p) return 0;
    const int K = (p->K >= 1 && p->K <= KBMOD_MAX_K) ? p->K : 1;
    const int TP = kb_padded_T(T);
    if (TP < 0) return 0;
    size_t o = align256(8 * sizeof(unsigned long long));
    // tables: offsets + the pruned plan's tables at their maximum group count
    const size_t ngm = std::min((size_t)n_vel, 2 * (((size_t)n_vel + 15) / 16) + 16);
    const size_t tiles_x = (W + 63) / 64, tiles_y = (H + 31) / 32;
    size_t tb = align256((size_t)n_vel * kb_tp4(TP) * 4) + align256((size_t)n_vel * 4) + align256(ngm * 16 * 4) + align256(ngm * (size_t)T * (16 * 4 + 32)) +
                align256(ngm * tiles_x * 8) + align256(ngm * tiles_y * 8) + align256(ngm * 4);
    o = align256(o + std::max<size_t>(tb, 256));
    o = align256(o + (size_t)H * W * K * 8);
    o = align256(o + (size_t)(3 * W) * (size_t)(3 * H) * (size_t)(T + 1) * 16);
    if (p->algo != KBMOD_ALGO_DIRECT) o = align256(o + kb_pruned_scratch_bytes(T, H, W, H, n_vel));
    return o;
}

static int search_rows(const float* d_psiphi, int T, int H, int W, const double* h_times, const float* h_vx,
                       const float* h_vy, int n_vel, const kbmod_search_params* p, int row_begin, int row_end, float* d_lh,
                       float* d_flux, int32_t* d_vel_idx, int32_t* d_n_obs, void* d_workspace, size_t workspace_bytes,
                       void* stream) {
    KB_REQUIRE(d_psiphi && h_times && p, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(row_begin == row_end || (d_lh && d_flux && d_vel_idx && d_n_obs), KBMOD_ERR_INVALID_ARG, "NULL argument");
    kbmod_plan* pl = nullptr;
    int rc = thread_plan(T, H, W, h_times, h_vx, h_vy, n_vel, p, row_begin, row_end, &pl);
    if (rc) return rc;
    return kbmod_plan_search(pl, d_psiphi, d_lh, d_flux, d_vel_idx, d_n_obs, d_workspace, workspace_bytes, stream);
}

extern "C" int kbmod_search(const float* d_psiphi, int T, int H, int W, const double* h_times, const float* h_vx,
                            const float* h_vy, int n_vel, const kbmod_search_params* p, float* d_lh, float* d_flux,
                            int32_t* d_vel_idx, int32_t* d_n_obs, void* d_workspace, size_t workspace_bytes,
                            void* stream) {
    return search_rows(d_psiphi, T, H, W, h_times, h_vx, h_vy, n_vel, p, 0, H, d_lh, d_flux, d_vel_idx, d_n_obs,
                       d_workspace, workspace_bytes, stream);
}

extern "C" int kbmod_search_rows(const float* d_psiphi, int T, int H, int W, const double* h_times, const float* h_vx,
                                 const float* h_vy, int n_vel, const kbmod_search_params* p, int row_begin, int row_end,
                                 float* d_lh, float* d_flux, int32_t* d_vel_idx, int32_t* d_n_obs, void* d_workspace,
                                 size_t workspace_bytes, void* stream) {
    return search_rows(d_psiphi, T, H, W, h_times, h_vx, h_vy, n_vel, p, row_begin, row_end, d_lh, d_flux, d_vel_idx,
                       d_n_obs, d_workspace, workspace_bytes, stream);
}

extern "C" int kbmod_search_unfiltered_lh(const void* d_workspace, const int32_t* d_vel_idx, float* d_lh_raw, void* stream) {
    KB_REQUIRE(g_plan, KBMOD_ERR_INVALID_ARG, "no kbmod_search on this thread yet");
    return kbmod_plan_unfiltered_lh(g_plan, d_workspace, d_vel_idx, d_lh_raw, stream);
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
    PrunedPlan pr;
    rc = kb_pruned_plan_build(T, H, W, 0, H, hdx.data(), hdy.data(), n_vel, &pr);
    if (rc) return rc;
    h_out[0] = (double)pr.too_scattered;
    h_out[1] = pr.evals > 0 ? pr.staged / pr.evals : 0.0;
    h_out[2] = (double)pr.ng;
    h_out[3] = pr.off_image;
    return KBMOD_OK;
}

extern "C" int kbmod_search_stats(const void* d_workspace, unsigned long long* h_out) {
    KB_REQUIRE(d_workspace && h_out, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_CUDA(cudaMemcpy(h_out, d_workspace, 5 * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    return KBMOD_OK;
}

// everything the library keeps per host thread: the cached plan of kbmod_search, the events of the phase timing,
// the copy streams and events of kbmod_pipeline_host_batch.  Safe to call at any time; the next call recreates
// what it needs.
static void release_batch_streams();
extern "C" int kbmod_release_thread_state(void) {
    kbmod_plan_destroy(g_plan);
    g_plan = nullptr;
    for (auto& m : g_marks) cudaEventDestroy(m.ev);
    g_marks.clear();
    for (auto& e : g_pool) cudaEventDestroy(e);
    g_pool.clear();
    release_batch_streams();
    cudaGetLastError();
    return KBMOD_OK;
}

// ---------------------------------------------------------------------------------------------
static const double kPaperMomentThr[5] = {0.5, 0.5, 1.5, 36.5, 36.5};

extern "C" int kbmod_coadd_stamps_filtered(const float* d_img, const uint8_t* d_mask, int T, int H, int W,
                                           const double* h_times, const int32_t* d_x0, const int32_t* d_y0,
                                           const float* d_vx, const float* d_vy, const uint64_t* d_epoch_mask, int n_traj,
                                           int radius, float* d_mean, float* d_median, const double* h_thresholds,
                                           double* d_moments, uint8_t* d_keep, void* stream) {
    KB_REQUIRE(d_img && h_times, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n_traj >= 0, KBMOD_ERR_INVALID_ARG, "n_traj = %d", n_traj);
    int rc = check_stack(T, H, W);
    if (rc) return rc;
    KB_REQUIRE(radius >= 0, KBMOD_ERR_INVALID_ARG, "radius = %d", radius);
    KB_REQUIRE(radius <= KBMOD_MAX_STAMP_RADIUS, KBMOD_ERR_UNSUPPORTED, "radius = %d exceeds %d", radius,
               KBMOD_MAX_STAMP_RADIUS);
    if (n_traj == 0 || (!d_mean && !d_median && !d_moments && !d_keep)) return KBMOD_OK;
    KB_REQUIRE(d_x0 && d_y0 && d_vx && d_vy, KBMOD_ERR_INVALID_ARG, "NULL trajectory arrays");
    if (h_thresholds)
        for (int k = 0; k < 5; ++k) KB_REQUIRE(!isnan(h_thresholds[k]), KBMOD_ERR_INVALID_ARG, "NaN threshold");
    const int TP = kb_padded_T(T);
    DevTimes times;
    make_times(h_times, T, &times);
    return kb_launch_coadd(d_img, d_mask, T, TP, H, W, times, d_x0, d_y0, d_vx, d_vy,
                           (const unsigned long long*)d_epoch_mask, n_traj, radius, d_mean, d_median,
                           h_thresholds ? h_thresholds : kPaperMomentThr, d_moments, d_keep, (cudaStream_t)stream);
}

extern "C" int kbmod_coadd_stamps(const float* d_img, const uint8_t* d_mask, int T, int H, int W,
                                  const double* h_times, const int32_t* d_x0, const int32_t* d_y0, const float* d_vx,
                                  const float* d_vy, const uint64_t* d_epoch_mask, int n_traj, int radius,
                                  float* d_mean, float* d_median, void* stream) {
    return kbmod_coadd_stamps_filtered(d_img, d_mask, T, H, W, h_times, d_x0, d_y0, d_vx, d_vy, d_epoch_mask, n_traj, radius,
                                       d_mean, d_median, nullptr, nullptr, nullptr, stream);
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
    return kbmod_sigmag_postfilter(d_psi_lc, d_phi_lc, n_lc, T, p, d_kept, d_lh, d_flux, nullptr, nullptr, nullptr, stream);
}

extern "C" int kbmod_sigmag_postfilter(const float* d_psi_lc, const float* d_phi_lc, int n_lc, int T,
                                       const kbmod_search_params* p, uint64_t* d_kept, float* d_lh, float* d_flux,
                                       uint8_t* d_pass, int32_t* d_survivors, uint64_t* d_n_pass, void* stream) {
    KB_REQUIRE(p, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n_lc >= 0, KBMOD_ERR_INVALID_ARG, "n_lc = %d", n_lc);
    KB_REQUIRE(!(d_survivors && !d_n_pass) && !(d_n_pass && !d_pass), KBMOD_ERR_INVALID_ARG,
               "d_survivors needs d_n_pass, and d_n_pass needs d_pass");
    if (d_n_pass) KB_CUDA(cudaMemsetAsync(d_n_pass, 0, 4 * sizeof(unsigned long long), (cudaStream_t)stream));
    kbmod_search_params q = *p;
    if (q.K < 1 || q.K > KBMOD_MAX_K) q.K = 1;
    DevParams P;
    int rc = kb_make_dev_params(&q, T, &P);
    if (rc) return rc;
    if (n_lc == 0) return KBMOD_OK;
    KB_REQUIRE(d_psi_lc && d_phi_lc, KBMOD_ERR_INVALID_ARG, "NULL lightcurves");
    return kb_launch_sigmag_filter(d_psi_lc, d_phi_lc, n_lc, T, kb_padded_T(T), P, (unsigned long long*)d_kept, d_lh,
                                   d_flux, d_pass, (unsigned long long*)d_n_pass, d_survivors, (cudaStream_t)stream);
}

extern "C" int kbmod_stamp_moments(const float* d_stamps, int n_stamps, int radius, const double* h_thresholds,
                                   double* d_moments, uint8_t* d_keep, void* stream) {
    KB_REQUIRE(n_stamps >= 0, KBMOD_ERR_INVALID_ARG, "n_stamps = %d", n_stamps);
    KB_REQUIRE(radius >= 0, KBMOD_ERR_INVALID_ARG, "radius = %d", radius);
    KB_REQUIRE(radius <= KBMOD_MAX_STAMP_RADIUS, KBMOD_ERR_UNSUPPORTED, "radius = %d exceeds %d", radius,
               KBMOD_MAX_STAMP_RADIUS);
    if (n_stamps == 0 || (!d_moments && !d_keep)) return KBMOD_OK;
    KB_REQUIRE(d_stamps, KBMOD_ERR_INVALID_ARG, "NULL stamps");
    if (h_thresholds)
        for (int k = 0; k < 5; ++k) KB_REQUIRE(!isnan(h_thresholds[k]), KBMOD_ERR_INVALID_ARG, "NaN threshold");
    return kb_launch_stamp_moments(d_stamps, n_stamps, radius, h_thresholds ? h_thresholds : kPaperMomentThr, d_moments, d_keep,
                                   (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------------------
// whole path from host buffers (bench.py's end-to-end number)
struct ArenaPlan {
    size_t off_img, off_var, off_mask, off_psiphi, off_lh, off_flux, off_vel, off_nobs, off_ws, ws_bytes, total;
};

static void plan_arena(int T, int H, int W, int K, size_t ws_bytes, ArenaPlan* a) {
    const size_t px = (size_t)T * H * W, res = (size_t)H * W * K;
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
    a->ws_bytes = ws_bytes;
    a->total = align256(o + ws_bytes);
}

extern "C" size_t kbmod_pipeline_host_arena_bytes(int T, int H, int W, int n_vel, const kbmod_search_params* p) {
    if (!p || T < 1 || T > KBMOD_MAX_T || H < 1 || W < 1 || n_vel < 0 || p->K < 1 || p->K > KBMOD_MAX_K) return 0;
    ArenaPlan a;
    plan_arena(T, H, W, p->K, kbmod_search_workspace_bytes(T, H, W, n_vel, p), &a);
    return a.total;
}

extern "C" size_t kbmod_pipeline_host_arena_bytes_for(int T, int H, int W, const double* h_times, const float* h_vx,
                                                      const float* h_vy, int n_vel, const kbmod_search_params* p) {
    if (!p || T < 1 || T > KBMOD_MAX_T || H < 1 || W < 1 || n_vel < 0 || p->K < 1 || p->K > KBMOD_MAX_K) return 0;
    const size_t ws = kbmod_search_workspace_bytes_for(T, H, W, h_times, h_vx, h_vy, n_vel, p, 0, H);
    if (!ws) return 0;
    ArenaPlan a;
    plan_arena(T, H, W, p->K, ws, &a);
    return a.total;
}

extern "C" int kbmod_pipeline_host(const float* h_img, const float* h_var, const uint8_t* h_mask, int T, int H, int W,
                                   const float* h_psf, int n_psf, int k, const double* h_times, const float* h_vx,
                                   const float* h_vy, int n_vel, const kbmod_search_params* p, float* h_lh,
                                   float* h_flux, int32_t* h_vel_idx, int32_t* h_n_obs, void* d_arena,
                                   size_t arena_bytes, void* stream) {
    const float* imgs[1] = {h_img};
    const float* vars[1] = {h_var};
    const uint8_t* masks[1] = {h_mask};
    float* lh[1] = {h_lh};
    float* fl[1] = {h_flux};
    int32_t* ve[1] = {h_vel_idx};
    int32_t* no[1] = {h_n_obs};
    return kbmod_pipeline_host_batch(1, imgs, vars, h_mask ? masks : nullptr, T, H, W, h_psf, n_psf, k, h_times, h_vx, h_vy,
                                     n_vel, p, lh, fl, ve, no, d_arena, arena_bytes, stream);
}

// ---------------------------------------------------------------------------------------------
// a batch of stacks of one shape (the CCDs of a pointing group): copies overlap the searches.  The two copy
// streams and six events are per host thread and per device; kbmod_release_thread_state() destroys them.
struct BatchStreams {
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t in_done[2] = {nullptr, nullptr}, comp_done[2] = {nullptr, nullptr}, out_done[2] = {nullptr, nullptr};
    bool ready = false;
    int device = -1;
};
static thread_local BatchStreams g_bs;

static void release_batch_streams() {
    if (!g_bs.ready) return;
    int cur = -1;
    cudaGetDevice(&cur);
    if (cur != g_bs.device) cudaSetDevice(g_bs.device);
    cudaStreamDestroy(g_bs.s_in);
    cudaStreamDestroy(g_bs.s_out);
    for (int b = 0; b < 2; ++b) {
        cudaEventDestroy(g_bs.in_done[b]);
        cudaEventDestroy(g_bs.comp_done[b]);
        cudaEventDestroy(g_bs.out_done[b]);
    }
    if (cur != g_bs.device && cur >= 0) cudaSetDevice(cur);
    g_bs = BatchStreams();
}

static int batch_body(int n_stacks, const float* const* h_img, const float* const* h_var, const uint8_t* const* h_mask,
                      int T, int H, int W, const float* h_psf, int n_psf, int k, kbmod_plan* pl, const ArenaPlan& a,
                      float* const* h_lh, float* const* h_flux, int32_t* const* h_vel_idx, int32_t* const* h_n_obs,
                      void* d_arena, cudaStream_t st) {
    const size_t px = (size_t)T * H * W, res = (size_t)H * W * pl->P.K;
    // everything enqueued on `stream` before this call happens-before the first copy
    // the plan's tables go into the workspace of each arena half once, before the first input copy is queued
    for (int b = 0; b < (n_stacks > 1 ? 2 : 1); ++b) {
        const int rcu = plan_upload_tables(pl, (char*)d_arena + (size_t)b * a.total + a.off_ws, st);
        if (rcu) return rcu;
    }
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
        int rc = kbmod_prepare_psi_phi((const float*)(A + a.off_img), (const float*)(A + a.off_var),
                                       hm ? (const uint8_t*)(A + a.off_mask) : nullptr, T, H, W, h_psf, n_psf, k,
                                       (float*)(A + a.off_psiphi), st);
        if (rc) return rc;
        rc = plan_search_impl(pl, (const float*)(A + a.off_psiphi), (float*)(A + a.off_lh), (float*)(A + a.off_flux),
                              (int32_t*)(A + a.off_vel), (int32_t*)(A + a.off_nobs), A + a.off_ws, a.ws_bytes, st, false);
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
    return KBMOD_OK;
}

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
    kbmod_plan* pl = nullptr;
    rc = thread_plan(T, H, W, h_times, h_vx, h_vy, n_vel, p, 0, H, &pl);
    if (rc) return rc;
    ArenaPlan a;
    plan_arena(T, H, W, p->K, pl->w_total, &a);
    const int n_buf = n_stacks > 1 ? 2 : 1;
    KB_REQUIRE(arena_bytes >= (size_t)n_buf * a.total, KBMOD_ERR_WORKSPACE,
               "arena of %zu bytes is smaller than the %d x %zu needed", arena_bytes, n_buf, a.total);
    for (int i = 0; i < n_stacks; ++i)
        KB_REQUIRE(h_img[i] && h_var[i] && h_lh[i] && h_flux[i] && h_vel_idx[i] && h_n_obs[i] && (!h_mask || h_mask[i]),
                   KBMOD_ERR_INVALID_ARG, "NULL buffer of stack %d", i);
    int dev = -1;
    KB_CUDA(cudaGetDevice(&dev));
    if (g_bs.ready && g_bs.device != dev) release_batch_streams();  // the thread moved to another GPU
    if (!g_bs.ready) {
        KB_CUDA(cudaStreamCreateWithFlags(&g_bs.s_in, cudaStreamNonBlocking));
        KB_CUDA(cudaStreamCreateWithFlags(&g_bs.s_out, cudaStreamNonBlocking));
        for (int b = 0; b < 2; ++b) {
            KB_CUDA(cudaEventCreateWithFlags(&g_bs.in_done[b], cudaEventDisableTiming));
            KB_CUDA(cudaEventCreateWithFlags(&g_bs.comp_done[b], cudaEventDisableTiming));
            KB_CUDA(cudaEventCreateWithFlags(&g_bs.out_done[b], cudaEventDisableTiming));
        }
        g_bs.ready = true;
        g_bs.device = dev;
    }
    cudaStream_t st = (cudaStream_t)stream;
    rc = batch_body(n_stacks, h_img, h_var, h_mask, T, H, W, h_psf, n_psf, k, pl, a, h_lh, h_flux, h_vel_idx, h_n_obs,
                    d_arena, st);
    // on success and on every error path alike: nothing of this call may still be reading or writing the caller's
    // host buffers when it returns
    const cudaError_t e1 = cudaStreamSynchronize(g_bs.s_in), e2 = cudaStreamSynchronize(st),
                      e3 = cudaStreamSynchronize(g_bs.s_out);
    if (rc) return rc;
    KB_CUDA(e1);
    KB_CUDA(e2);
    KB_CUDA(e3);
    return KBMOD_OK;
}
