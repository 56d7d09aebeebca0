/*
 * oracle/kbmod_oracle.c  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU restatement of what the KBMOD shift-and-stack hot path
 * computes, written from the paper (arXiv 2109.03296, /root/reference/PAPER.md) and from the
 * readings DESIGN.md lists where the paper is silent.  It shares no code, header, table or
 * constant generator with the CUDA library under paper_2109_03296_b200/csrc and neither
 * includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * Precision: sums, scores, convolutions and stamp statistics are IEEE double.  The one place
 * where floating point decides an integer -- the sigma-G kept set (which epochs survive the
 * clip) -- is taken in IEEE single, the kernel's precision, with every operation separately
 * rounded (build with -ffp-contract=off), as the task's parity rules require for decisions.
 *
 * Steps (names follow SURVEY.md section 8c):
 *   O1 psi/phi preparation     PAPER.md L79  (section 3; Whidden et al. 2019 matched filter)
 *   O2 displacement table      PAPER.md L79-L81 ("shifted along a potential asteroid trajectory")
 *   O3 gather along trajectory PAPER.md L79  (Psi_coadd = sum Psi_i, Phi_coadd = sum Phi_i)
 *   O4 sigma-G filter          PAPER.md L95-L117 (section 3.1, Eq. 1-5)
 *   O5 score                   PAPER.md L79  (nu = Psi_coadd / sqrt(Phi_coadd)), L123 (sum LH')
 *   O6 per-pixel top-K         PAPER.md L127-L137 (section 3.2)
 *   O7 coadded stamps          PAPER.md L141 (section 3.3), L131 (Fig. 5)
 *   N2 stamp central moments   PAPER.md L141 (section 3.3): thresholds 0.5, 0.5, 1.5, 36.5, 36.5; reading R22
 *
 * Pins (tests/test_oracle_*.py): closed-form point source, all-zero psi, numpy brute force on
 * tiny stacks, sorted() percentiles, erf^-1 closed form of the 0.7413 coefficient, invariants.
 * Interpolated percentiles (R23) are pinned against numpy.percentile(method="linear"); the unfiltered sum-LH
 * against the sigma-G-off evaluation; the post-filter's reject flag against the paper's threshold (L123).
 * Unpinned against the original KBMOD code (not available): readings R3 (masked taps), R10
 * (nearest-rank percentiles) and R22 (moment normalisation) -- "parity unpinned" with respect to that
 * code; see DESIGN.md.
 */
#include <float.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#if defined(FLT_EVAL_METHOD) && FLT_EVAL_METHOD != 0
#error "single-precision decisions need FLT_EVAL_METHOD == 0 (SSE arithmetic)"
#endif

#define ORACLE_MAX_T 64

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* number of OpenMP threads the following calls use (bench.py's 1-core baseline figure); no arithmetic here */
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------ O1: psi / phi (L79; R1-R4) */
static int pixel_good(const float *img, const float *var, const uint8_t *mask, int H, int W, int y, int x) {
    if (x < 0 || x >= W || y < 0 || y >= H) return 0;
    size_t i = (size_t)y * W + x;
    if (mask && mask[i] != 0) return 0;
    if (!(var[i] > 0.0f) || !isfinite(var[i]) || !isfinite(img[i])) return 0;
    return 1;
}

/* Psi = sum_{j,i} P[j][i] * I(x+i-r, y+j-r) * w,  Phi = sum P[j][i]^2 * w,  w = 1/var for good
 * pixels and 0 otherwise (correlation, no kernel flip, no renormalisation).  An output pixel is
 * invalid (psi = phi = 0, valid = 0) iff its own centre pixel is bad.  psi_abs (nullable) gets
 * sum |P I w|, the scale a float32 comparison tolerance is relative to. */
void oracle_prepare_psi_phi(const float *img, const float *var, const uint8_t *mask, int T, int H, int W,
                            const float *psf, int n_psf, int k, double *psi, double *phi, uint8_t *valid,
                            double *psi_abs) {
    const int r = k / 2;
    const size_t plane = (size_t)H * W;
    for (int t = 0; t < T; ++t) {
        const float *I = img + t * plane, *V = var + t * plane;
        const uint8_t *M = mask ? mask + t * plane : NULL;
        const float *P = psf + (n_psf > 1 ? (size_t)t * k * k : 0);
#pragma omp parallel for schedule(static)
        for (int y = 0; y < H; ++y) {
            for (int x = 0; x < W; ++x) {
                size_t o = t * plane + (size_t)y * W + x;
                if (!pixel_good(I, V, M, H, W, y, x)) {
                    psi[o] = 0.0; phi[o] = 0.0; valid[o] = 0;
                    if (psi_abs) psi_abs[o] = 0.0;
                    continue;
                }
                double sp = 0.0, sf = 0.0, sa = 0.0;
                for (int j = 0; j < k; ++j)
                    for (int i = 0; i < k; ++i) {
                        int xx = x + i - r, yy = y + j - r;
                        if (!pixel_good(I, V, M, H, W, yy, xx)) continue;
                        size_t q = (size_t)yy * W + xx;
                        double w = 1.0 / (double)V[q];
                        double p = (double)P[j * k + i];
                        sp += p * (double)I[q] * w;
                        sa += fabs(p * (double)I[q] * w);
                        sf += p * p * w;
                    }
                psi[o] = sp; phi[o] = sf; valid[o] = 1;
                if (psi_abs) psi_abs[o] = sa;
            }
        }
    }
}

/* ------------------------------------------------------------------ O2: displacements (R5, R18) */
/* d = floor(v * (t - t0) + 1/2), round-half-up, in double; multiply and add separately rounded. */
static int32_t displacement(float v, double dt) {
    double p = (double)v * dt;
    double q = p + 0.5;
    return (int32_t)floor(q);
}

void oracle_displacements(const double *times, int T, const float *vx, const float *vy, int n_vel,
                          int32_t *dx, int32_t *dy) {
    for (int v = 0; v < n_vel; ++v)
        for (int t = 0; t < T; ++t) {
            double dt = times[t] - times[0];
            dx[(size_t)v * T + t] = displacement(vx[v], dt);
            dy[(size_t)v * T + t] = displacement(vy[v], dt);
        }
}

/* ------------------------------------------------------------------ O4: sigma-G (L95-L117; R9-R13) */
typedef struct {
    int sigmag_enable;
    float pct_lo, pct_hi, coeff, n_sigma;
    int filter_on; /* 0: flux psi/phi, 1: likelihood psi/sqrt(phi)  (L123 "likelihood and/or flux") */
    float min_lh;
    int min_obs, K;
    int pct_interp; /* 0: nearest-rank order statistics (R10); 1: linear interpolation between them (R23) */
} oparams;

/* nearest-rank percentile index: ceil(q n / 100) - 1, clamped to [0, n-1]  (R10) */
static int pct_rank(float q, int n) {
    int r = (int)ceil((double)q * (double)n / 100.0) - 1;
    if (r < 0) r = 0;
    if (r > n - 1) r = n - 1;
    return r;
}

int oracle_pct_rank(float q, int n) { return pct_rank(q, n); }

/* The q-th percentile of the ascending array s[0..m).  PAPER.md L117: "selecting the 25th and 75th percentile
 * values ... from the data".  interp = 0 (reading R10, the default): the nearest-rank order statistic.
 * interp = 1 (reading R23, the alternative SURVEY 8c-R10 names): linear interpolation between the two order
 * statistics that bracket the fractional position h = (m - 1) q / 100,
 *     v = s[k] + g (s[k+1] - s[k]),   k = floor(h),  g = h - k,
 * h and g in double, g rounded to single, then the three single-precision operations separately rounded
 * (the decision precision).  This is numpy.percentile(method="linear") up to single-precision rounding. */
static float pct_value(const float *s, int m, float q, int interp) {
    if (!interp) return s[pct_rank(q, m)];
    double h = (double)(m - 1) * (double)q / 100.0;
    if (h <= 0.0) return s[0];
    if (h >= (double)(m - 1)) return s[m - 1];
    int k = (int)floor(h);
    float g = (float)(h - (double)k);
    float d = s[k + 1] - s[k];
    float e = g * d;
    return s[k] + e;
}

float oracle_pct_value(const float *s, int m, float q, int interp) { return pct_value(s, m, q, interp); }

/* psi_t, phi_t: the T gathered samples; valid: bit t set iff epoch t contributes.
 * Returns n_kept (0 = "no result": fewer than max(1, min_obs) valid epochs). */
static int filter_and_score(const float *psi_t, const float *phi_t, int T, uint64_t valid, const oparams *p,
                            uint64_t *kept_out, double *lh, double *flux) {
    int n = 0;
    for (int t = 0; t < T; ++t) n += (int)((valid >> t) & 1u);
    int need = p->min_obs > 1 ? p->min_obs : 1;
    *kept_out = 0; *lh = -INFINITY; *flux = 0.0;
    if (n < need) return 0;

    uint64_t kept = valid;
    if (p->sigmag_enable) {
        float f[ORACLE_MAX_T], s[ORACLE_MAX_T];
        int m = 0;
        for (int t = 0; t < T; ++t) {
            if (!((valid >> t) & 1u)) continue;
            /* single precision, correctly rounded: the decision precision */
            f[t] = p->filter_on ? psi_t[t] / sqrtf(phi_t[t]) : psi_t[t] / phi_t[t];
            s[m++] = f[t];
        }
        for (int i = 1; i < m; ++i) { /* insertion sort, ascending */
            float key = s[i];
            int j = i - 1;
            while (j >= 0 && s[j] > key) { s[j + 1] = s[j]; --j; }
            s[j + 1] = key;
        }
        float p_lo = pct_value(s, m, p->pct_lo, p->pct_interp);
        float p_50 = pct_value(s, m, 50.0f, p->pct_interp);
        float p_hi = pct_value(s, m, p->pct_hi, p->pct_interp);
        float d = p_hi - p_lo;       /* Eq. 5: sigma_G = C (x_j - x_i) */
        float sg = p->coeff * d;
        float w = p->n_sigma * sg;   /* L117: +- n sigma_G about the median */
        float lo = p_50 - w;
        float hi = p_50 + w;
        kept = 0;
        for (int t = 0; t < T; ++t)
            if (((valid >> t) & 1u) && f[t] >= lo && f[t] <= hi) kept |= (uint64_t)1 << t;
    }
    /* O5: recompute sum LH' from the survivors (L123), double precision */
    double sp = 0.0, sf = 0.0;
    int nk = 0;
    for (int t = 0; t < T; ++t)
        if ((kept >> t) & 1u) { sp += (double)psi_t[t]; sf += (double)phi_t[t]; ++nk; }
    *kept_out = kept;
    *lh = sp / sqrt(sf);
    *flux = sp / sf;
    return nk;
}

/* O3: gather the T samples of one trajectory.  psiphi is [T][H][W][2] float (psi, phi interleaved);
 * a sample is valid iff on-image and phi > 0 (the invalid encoding is psi = phi = 0). */
static uint64_t gather(const float *psiphi, int T, int H, int W, int x0, int y0, const int32_t *dx,
                       const int32_t *dy, float *psi_t, float *phi_t) {
    uint64_t valid = 0;
    const size_t plane = (size_t)H * W;
    for (int t = 0; t < T; ++t) {
        int x = x0 + dx[t], y = y0 + dy[t];
        psi_t[t] = 0.0f; phi_t[t] = 0.0f;
        if (x < 0 || x >= W || y < 0 || y >= H) continue;
        const float *q = psiphi + 2 * (t * plane + (size_t)y * W + x);
        if (!(q[1] > 0.0f)) continue;
        psi_t[t] = q[0]; phi_t[t] = q[1];
        valid |= (uint64_t)1 << t;
    }
    return valid;
}

/* ------------------------------------------------------------------ O3-O6: search over a pixel list */
/* For every listed start pixel and every velocity: gather, filter, score, threshold (L' >= min_lh),
 * and keep the K best per pixel ordered by (L' descending, vel_idx ascending).  Unfilled slots:
 * lh = -inf, flux = 0, vel_idx = -1, n_obs = 0.  Outputs are [n_pix][K]. */
void oracle_search_pixels(const float *psiphi, int T, int H, int W, const double *times, const float *vx,
                          const float *vy, int n_vel, const int32_t *px, const int32_t *py, int n_pix,
                          int sigmag_enable, float pct_lo, float pct_hi, float coeff, float n_sigma,
                          int filter_on, float min_lh, int min_obs, int K, int pct_interp, double *lh, double *flux,
                          int32_t *vel_idx, int32_t *n_obs) {
    oparams p = {sigmag_enable, pct_lo, pct_hi, coeff, n_sigma, filter_on, min_lh, min_obs, K, pct_interp};
    int32_t *dx = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_vel * T);
    int32_t *dy = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_vel * T);
    oracle_displacements(times, T, vx, vy, n_vel, dx, dy);
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < n_pix; ++i) {
        double *L = lh + (size_t)i * K, *F = flux + (size_t)i * K;
        int32_t *V = vel_idx + (size_t)i * K, *N = n_obs + (size_t)i * K;
        for (int k = 0; k < K; ++k) { L[k] = -INFINITY; F[k] = 0.0; V[k] = -1; N[k] = 0; }
        float psi_t[ORACLE_MAX_T], phi_t[ORACLE_MAX_T];
        for (int v = 0; v < n_vel; ++v) {
            uint64_t valid = gather(psiphi, T, H, W, px[i], py[i], dx + (size_t)v * T, dy + (size_t)v * T,
                                    psi_t, phi_t);
            uint64_t kept; double l, f;
            int nk = filter_and_score(psi_t, phi_t, T, valid, &p, &kept, &l, &f);
            if (nk == 0) continue;
            if (!(l >= (double)min_lh)) continue; /* R14 */
            /* O6: insert; velocities arrive in ascending index, so strict > keeps lower index first */
            int pos = K;
            while (pos > 0 && (V[pos - 1] < 0 || l > L[pos - 1])) --pos;
            if (pos >= K) continue;
            for (int k = K - 1; k > pos; --k) { L[k] = L[k - 1]; F[k] = F[k - 1]; V[k] = V[k - 1]; N[k] = N[k - 1]; }
            L[pos] = l; F[pos] = f; V[pos] = v; N[pos] = nk;
        }
    }
    free(dx); free(dy);
}

/* ------------------------------------------------------------------ single-trajectory variant (L175) */
/* Reports L', flux' regardless of min_lh.  n_valid < max(1, min_obs): lh = -inf, flux = 0, kept = 0. */
void oracle_eval_trajectories(const float *psiphi, int T, int H, int W, const double *times, const int32_t *x0,
                              const int32_t *y0, const float *vx, const float *vy, int n_traj,
                              int sigmag_enable, float pct_lo, float pct_hi, float coeff, float n_sigma,
                              int filter_on, int min_obs, int pct_interp, float *psi_lc, float *phi_lc,
                              uint64_t *valid_out, uint64_t *kept_out, double *lh, double *flux, int32_t *n_kept) {
    oparams p = {sigmag_enable, pct_lo, pct_hi, coeff, n_sigma, filter_on, -INFINITY, min_obs, 1, pct_interp};
#pragma omp parallel for schedule(dynamic, 64)
    for (int i = 0; i < n_traj; ++i) {
        int32_t dx[ORACLE_MAX_T], dy[ORACLE_MAX_T];
        oracle_displacements(times, T, vx + i, vy + i, 1, dx, dy);
        float *ps = psi_lc + (size_t)i * T, *ph = phi_lc + (size_t)i * T;
        uint64_t valid = gather(psiphi, T, H, W, x0[i], y0[i], dx, dy, ps, ph);
        valid_out[i] = valid;
        n_kept[i] = filter_and_score(ps, ph, T, valid, &p, &kept_out[i], &lh[i], &flux[i]);
    }
}

/* sigma-G on given lightcurves [n_lc][T] (config 5's "rerun sigma-G"); valid iff phi > 0.
 * The paper's post-filter: "reject the trajectory if the recomputed likelihood (sum LH') is
 * less than 10": pass[i] = 1 iff the lightcurve has a result (n_valid >= max(1, min_obs)) and L' >= min_lh
 * (reading R14: the comparison is >=; min_lh = -inf keeps every lightcurve that has a result). */
void oracle_sigmag_filter(const float *psi_lc, const float *phi_lc, int n_lc, int T, int sigmag_enable,
                          float pct_lo, float pct_hi, float coeff, float n_sigma, int filter_on, int min_obs,
                          int pct_interp, float min_lh, uint64_t *kept_out, double *lh, double *flux,
                          int32_t *n_kept, uint8_t *pass) {
    oparams p = {sigmag_enable, pct_lo, pct_hi, coeff, n_sigma, filter_on, -INFINITY, min_obs, 1, pct_interp};
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n_lc; ++i) {
        const float *ps = psi_lc + (size_t)i * T, *ph = phi_lc + (size_t)i * T;
        uint64_t valid = 0;
        for (int t = 0; t < T; ++t)
            if (ph[t] > 0.0f) valid |= (uint64_t)1 << t;
        n_kept[i] = filter_and_score(ps, ph, T, valid, &p, &kept_out[i], &lh[i], &flux[i]);
        if (pass) pass[i] = (n_kept[i] > 0 && lh[i] >= (double)min_lh) ? 1 : 0;
    }
}

/* ------------------------------------------------------------------ unfiltered sum-LH beside sum-LH' (L175, L181) */
/* PAPER.md L175 (section 4.1): the single-trajectory variant "computes the likelihoods along a single trajectory
 * then runs the ... filtering"; L181 quotes the unfiltered sum-LH next to the filtered sum-LH' of recovered objects.
 * For every result slot (pixel i, slot k) with vel_idx >= 0: L = sum_valid psi / sqrt(sum_valid phi) over ALL
 * valid epochs of that trajectory (no sigma-G clip, no threshold), double precision; empty slots get -inf. */
void oracle_unfiltered_lh(const float *psiphi, int T, int H, int W, const double *times, const float *vx,
                          const float *vy, int n_vel, const int32_t *px, const int32_t *py, int n_pix, int K,
                          const int32_t *vel_idx, double *lh_raw) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int i = 0; i < n_pix; ++i)
        for (int k = 0; k < K; ++k) {
            int v = vel_idx[(size_t)i * K + k];
            double *out = lh_raw + (size_t)i * K + k;
            *out = -INFINITY;
            if (v < 0 || v >= n_vel) continue;
            int32_t dx[ORACLE_MAX_T], dy[ORACLE_MAX_T];
            float psi_t[ORACLE_MAX_T], phi_t[ORACLE_MAX_T];
            oracle_displacements(times, T, vx + v, vy + v, 1, dx, dy);
            uint64_t valid = gather(psiphi, T, H, W, px[i], py[i], dx, dy, psi_t, phi_t);
            double sp = 0.0, sf = 0.0;
            for (int t = 0; t < T; ++t)
                if ((valid >> t) & 1u) { sp += (double)psi_t[t]; sf += (double)phi_t[t]; }
            if (valid) *out = sp / sqrt(sf);
        }
}

/* ------------------------------------------------------------------ O7: coadded stamps (L141; R17) */
/* For each trajectory and stamp offset (u, v) in [-r, r]^2: the samples are the image-plane pixels
 * I_t(x0 + dx_t + u, y0 + dy_t + v) of the selected epochs that are on-image, unmasked and finite.
 * mean = sum / count; median = middle of the sort (mean of the two middles for an even count);
 * count 0 -> 0.  Outputs are [n_traj][2r+1][2r+1] (v rows, u columns). */
void oracle_coadd_stamps(const float *img, const uint8_t *mask, int T, int H, int W, const double *times,
                         const int32_t *x0, const int32_t *y0, const float *vx, const float *vy,
                         const uint64_t *epoch_mask, int n_traj, int radius, double *mean, double *median) {
    const int S = 2 * radius + 1;
    const size_t plane = (size_t)H * W;
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < n_traj; ++i) {
        int32_t dx[ORACLE_MAX_T], dy[ORACLE_MAX_T];
        oracle_displacements(times, T, vx + i, vy + i, 1, dx, dy);
        for (int v = -radius; v <= radius; ++v)
            for (int u = -radius; u <= radius; ++u) {
                double vals[ORACLE_MAX_T];
                int m = 0;
                for (int t = 0; t < T; ++t) {
                    if (epoch_mask && !((epoch_mask[i] >> t) & 1u)) continue;
                    int x = x0[i] + dx[t] + u, y = y0[i] + dy[t] + v;
                    if (x < 0 || x >= W || y < 0 || y >= H) continue;
                    size_t q = t * plane + (size_t)y * W + x;
                    if (mask && mask[q] != 0) continue;
                    if (!isfinite(img[q])) continue;
                    vals[m++] = (double)img[q];
                }
                double mu = 0.0, med = 0.0;
                if (m > 0) {
                    for (int a = 0; a < m; ++a) mu += vals[a];
                    mu /= (double)m;
                    for (int a = 1; a < m; ++a) {
                        double key = vals[a];
                        int b = a - 1;
                        while (b >= 0 && vals[b] > key) { vals[b + 1] = vals[b]; --b; }
                        vals[b + 1] = key;
                    }
                    med = (m & 1) ? vals[m / 2] : 0.5 * (vals[m / 2 - 1] + vals[m / 2]);
                }
                size_t o = ((size_t)i * S + (v + radius)) * S + (u + radius);
                if (mean) mean[o] = mu;
                if (median) median[o] = med;
            }
    }
}

/* ------------------------------------------------------------------ N2: central-moment stamp filter (L141) */
/* PAPER.md L141 (section 3.3): "we computed the central moments of postage stamps ... Stamps were rejected if they
 * did not have central moments that were consistent with a Gaussian ... we required that the x, y, xy, xx, and yy
 * moments be strictly less than 0.5, 0.5, 1.5, 36.5, and 36.5 respectively."  Reading R22: the stamp
 * is made non-negative by subtracting its minimum and normalised to unit sum, w = (I - min I) / sum(I - min I)
 * (a constant stamp gets the uniform weights 1/N); the moments are taken about the CENTRE PIXEL in pixel units,
 *     m_x = sum u w,  m_y = sum v w,  m_xy = sum u v w,  m_xx = sum u^2 w,  m_yy = sum v^2 w,   u, v in [-r, r];
 * the first three are compared by absolute value.  Non-finite pixels make the stamp fail.
 * Pin of the reading: a featureless stamp has m_xx = m_yy = r (r + 1) / 3 = 36.67 for the paper's 21x21 stamps,
 * just above the paper's 36.5 -- the thresholds reject "no source at all" only under this normalisation.
 * stamps [n][S][S] float (v rows, u columns), thr[5]; out: moments [n][5] double, pass [n] (1 = kept). */
void oracle_stamp_moments(const float *stamps, int n, int radius, const double *thr, double *moments, uint8_t *pass) {
    const int S = 2 * radius + 1, N = S * S;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n; ++i) {
        const float *I = stamps + (size_t)i * N;
        double *m = moments + (size_t)i * 5;
        int finite = 1;
        double mn = INFINITY;
        for (int k = 0; k < N; ++k) {
            if (!isfinite(I[k])) finite = 0;
            else if ((double)I[k] < mn) mn = (double)I[k];
        }
        if (!finite) { for (int k = 0; k < 5; ++k) m[k] = NAN; pass[i] = 0; continue; }
        double sum = 0.0;
        for (int k = 0; k < N; ++k) sum += (double)I[k] - mn;
        double mx = 0, my = 0, mxy = 0, mxx = 0, myy = 0;
        for (int v = -radius; v <= radius; ++v)
            for (int u = -radius; u <= radius; ++u) {
                double w = sum > 0.0 ? ((double)I[(v + radius) * S + (u + radius)] - mn) / sum : 1.0 / (double)N;
                mx += u * w; my += v * w; mxy += (double)(u * v) * w; mxx += (double)(u * u) * w; myy += (double)(v * v) * w;
            }
        m[0] = mx; m[1] = my; m[2] = mxy; m[3] = mxx; m[4] = myy;
        pass[i] = (fabs(mx) < thr[0] && fabs(my) < thr[1] && fabs(mxy) < thr[2] && mxx < thr[3] && myy < thr[4]) ? 1 : 0;
    }
}
