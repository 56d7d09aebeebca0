// Internal declarations shared by the kernels of libkbmod_b200.so.  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>
#include <stdio.h>

#include <vector>

#include "../../include/kbmod_b200.h"
#include "sortnet_gen.cuh"

// ---------------------------------------------------------------------------------------------
// errors
void kb_set_error(const char* fmt, ...);
#define KB_CUDA(call)                                                                            \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            kb_set_error("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return KBMOD_ERR_CUDA;                                                               \
        }                                                                                        \
    } while (0)
#define KB_REQUIRE(cond, code, ...)                                                              \
    do {                                                                                         \
        if (!(cond)) {                                                                           \
            kb_set_error(__VA_ARGS__);                                                           \
            return (code);                                                                       \
        }                                                                                        \
    } while (0)

// ---------------------------------------------------------------------------------------------
// parameters as the kernels see them (passed by value in the kernel parameter bank)
struct DevParams {
    int sigmag_enable, filter_on, min_obs, K, T, pct_interp;
    float coeff, n_sigma, min_lh;
    // percentiles of n valid samples, n = 0..64 ("selecting the 25th and 75th percentile values ...
    // from the data").  rk_*[n] = index k into the ascending sort; fr_*[n] < 0: the value is s[k] (nearest rank
    // ceil(q n / 100) - 1, reading R10; also the clamped ends of the interpolated form); fr_*[n] = g >= 0: the value
    // is s[k] + g (s[k+1] - s[k]), linear interpolation at h = (n - 1) q / 100 (reading R23)
    unsigned char rk_lo[KBMOD_MAX_T + 1], rk_md[KBMOD_MAX_T + 1], rk_hi[KBMOD_MAX_T + 1];
    float fr_lo[KBMOD_MAX_T + 1], fr_md[KBMOD_MAX_T + 1], fr_hi[KBMOD_MAX_T + 1];
};
struct DevTimes {
    double dt[KBMOD_MAX_T];  // times[t] - times[0]
};

int kb_make_dev_params(const kbmod_search_params* p, int T, DevParams* out);  // validates
int kb_padded_T(int T);  // smallest instantiated network size >= T, or -1

// ---------------------------------------------------------------------------------------------
// dispatch on the padded epoch count
#define KB_DISPATCH_TP(TPv, ...)                                                                 \
    switch (TPv) {                                                                               \
        case 4: { constexpr int TP = 4; __VA_ARGS__; } break;                                    \
        case 5: { constexpr int TP = 5; __VA_ARGS__; } break;                                    \
        case 8: { constexpr int TP = 8; __VA_ARGS__; } break;                                    \
        case 10: { constexpr int TP = 10; __VA_ARGS__; } break;                                  \
        case 12: { constexpr int TP = 12; __VA_ARGS__; } break;                                  \
        case 16: { constexpr int TP = 16; __VA_ARGS__; } break;                                  \
        case 20: { constexpr int TP = 20; __VA_ARGS__; } break;                                  \
        case 24: { constexpr int TP = 24; __VA_ARGS__; } break;                                  \
        case 26: { constexpr int TP = 26; __VA_ARGS__; } break;                                  \
        case 28: { constexpr int TP = 28; __VA_ARGS__; } break;                                  \
        case 32: { constexpr int TP = 32; __VA_ARGS__; } break;                                  \
        case 40: { constexpr int TP = 40; __VA_ARGS__; } break;                                  \
        case 48: { constexpr int TP = 48; __VA_ARGS__; } break;                                  \
        case 50: { constexpr int TP = 50; __VA_ARGS__; } break;                                  \
        case 56: { constexpr int TP = 56; __VA_ARGS__; } break;                                  \
        case 64: { constexpr int TP = 64; __VA_ARGS__; } break;                                  \
        default: kb_set_error("no kernel instantiated for padded T = %d", TPv); return KBMOD_ERR_UNSUPPORTED; \
    }

// ---------------------------------------------------------------------------------------------
// device: displacement (reading R5) -- the same two separately rounded double operations as the
// host table, so positions are bit-identical wherever they are computed.
__device__ __forceinline__ int kb_displacement(float v, double dt) {
    double p = __dmul_rn((double)v, dt);
    double q = __dadd_rn(p, 0.5);
    return (int)floor(q);
}

// device: one percentile from the ascending sort parked in shared memory (element k at scratch[k * stride])
__device__ __forceinline__ float kb_percentile(const float* scratch, int stride, int k, float g, int interp) {
    const float a = scratch[k * stride];
    if (!interp || g < 0.0f) return a;
    const float b = scratch[(k + 1) * stride];
    // float32, each operation separately rounded: the precision the keep/drop decision is taken in (R20, R23)
    const float d = __fsub_rn(b, a);
    const float e = __fmul_rn(g, d);
    return __fadd_rn(a, e);
}

// device: the clip window [lo, hi] of the sigma-G filter from the sorted lightcurve values s[0..n) (+inf behind them)
// PAPER.md:L95-L117 Eq. 1-5: sigma_G = C (P_hi - P_lo); keep points within +- n sigma_G of the median (L117)
template <int TP>
__device__ __forceinline__ void kb_clip_window(float (&s)[TP], int n, const DevParams& P, float* scratch, int stride,
                                               float& lo, float& hi) {
    SortNet<TP>::sort(s);  // invalid epochs (+inf) end up behind the n valid ones
#pragma unroll
    for (int t = 0; t < TP; ++t) scratch[t * stride] = s[t];
    const float p_lo = kb_percentile(scratch, stride, P.rk_lo[n], P.fr_lo[n], P.pct_interp);
    const float p_50 = kb_percentile(scratch, stride, P.rk_md[n], P.fr_md[n], P.pct_interp);
    const float p_hi = kb_percentile(scratch, stride, P.rk_hi[n], P.fr_hi[n], P.pct_interp);
    const float d = __fsub_rn(p_hi, p_lo);      // Eq. 5: sigma_G = C (x_j - x_i)
    const float sg = __fmul_rn(P.coeff, d);
    const float w = __fmul_rn(P.n_sigma, sg);   // L117: +- n sigma_G about the median
    lo = __fsub_rn(p_50, w);
    hi = __fadd_rn(p_50, w);
}

// the per-epoch value the filter works on (reading R9): flux psi/phi, or likelihood psi/sqrt(phi) with filter_on.
// IEEE float32, correctly rounded; the same two intrinsics wherever it is computed (per pixel in s4_build_kernel,
// per sample in the lightcurve kernels), so the filtered values are bit-identical on every path
__device__ __forceinline__ float kb_filter_value(float psi, float phi, int filter_on) {
    const float den = filter_on ? __fsqrt_rn(phi) : phi;
    return __fdiv_rn(psi, den);
}

// L' and flux' from the kept sums (nu = Psi_coadd / sqrt(Phi_coadd), recomputed from the survivors,
// L123).  One definition for every search kernel so that the direct and the pruned path return identical bits.
__device__ __forceinline__ float kb_lh_of(float sp, float sf) { return sp * rsqrtf(sf); }
__device__ __forceinline__ float kb_flux_of(float sp, float sf) { return __fdividef(sp, sf); }

// device: sigma-G filter + score of one lightcurve held in registers (steps 2-3 of kbmod_search;
// PAPER.md:L95-L117 Eq. 1-5).  Epoch t is valid iff phi[t] > 0.  General form: takes (psi, phi) only,
// reports the kept bitmap; used by the lightcurve kernels.
//   scratch: shared memory, this thread's column; element k lives at scratch[k * stride].
// Returns n_kept; 0 means "no result" (fewer than max(1,min_obs) valid epochs, or nothing kept).
template <int TP>
__device__ __forceinline__ int kb_score_lightcurve(const float (&psi)[TP], const float (&phi)[TP],
                                                   const DevParams& P, float* scratch, int stride, float& lh,
                                                   float& flux, unsigned long long& kept_mask) {
    int n = 0;
#pragma unroll
    for (int t = 0; t < TP; ++t) n += (phi[t] > 0.0f) ? 1 : 0;
    lh = -CUDART_INF_F;
    flux = 0.0f;
    kept_mask = 0ull;
    const int need = P.min_obs > 1 ? P.min_obs : 1;
    if (n < need) return 0;

    float f[TP];
    float lo = -CUDART_INF_F, hi = CUDART_INF_F;
    if (P.sigmag_enable) {
        float s[TP];
#pragma unroll
        for (int t = 0; t < TP; ++t) {
            // (an invalid epoch divides by zero and the result is discarded: guarding the operands instead was
            // measured 2-3 % slower once the warps stay converged)
            f[t] = (phi[t] > 0.0f) ? kb_filter_value(psi[t], phi[t], P.filter_on) : CUDART_INF_F;
            s[t] = f[t];
        }
        kb_clip_window<TP>(s, n, P, scratch, stride, lo, hi);
    } else {
#pragma unroll
        for (int t = 0; t < TP; ++t) f[t] = 0.0f;
    }
    float sp = 0.0f, sf = 0.0f;
    int nk = 0;
#pragma unroll
    for (int t = 0; t < TP; ++t) {
        const bool keep = (phi[t] > 0.0f) && (f[t] >= lo) && (f[t] <= hi);
        if (keep) {
            sp += psi[t];
            sf += phi[t];
            ++nk;
            kept_mask |= 1ull << t;
        }
    }
    if (nk == 0) return 0;
    lh = kb_lh_of(sp, sf);
    flux = kb_flux_of(sp, sf);
    return nk;
}

// ---------------------------------------------------------------------------------------------
// The search kernels' working copy of the psi/phi stack (the "canvas", built by s4_build_kernel at the start of
// every kbmod_search): one float2 per pixel of a padded canvas,
//     (f, m)   valid pixel:   f = kb_filter_value(psi, phi), the value the filter sorts and clips;
//                             m = MINUS the denominator f was divided by: -phi, or -sqrt(phi) with filter_on
//              invalid pixel, padding, and the extra plane T: (+inf, +0)
// padded by the largest displacement of the velocity list on each side (clamped to the image size), so a
// trajectory sample is ONE 8-byte load at  base(x0, y0) + off[v][t]  with no bounds test: off-image samples land
// in the padding and read "invalid".  Epochs t >= T of the padded count TP point into plane T.
// The kept sums are accumulated from these two numbers (reading R25): sum psi as fma(f, -m, sum) -- f |m| is
// psi up to two float32 roundings (1.2e-7 relative, against the 1e-4 the results are held to) -- and sum phi as
// sum - m, or fma(m, m, sum) with filter_on.  The sign bit of m is the valid flag, so counting the valid samples
// costs one shift-add per sample.  A warp's 32 samples of one epoch are 256 contiguous bytes (two or three lines)
// instead of the 512 of a (psi, phi, f, valid) cell, and a lightcurve occupies 2 x T registers instead of 3 x T.
struct S4Geom {
    int Wp, Hp;        // padded canvas
    int pxn, pyn;      // padding on the low-x / low-y side (image pixel (x, y) sits at (x + pxn, y + pyn))
    unsigned int plane;  // Wp * Hp
};
__host__ __device__ inline int kb_tp4(int TP) { return (TP + 3) & ~3; }

// gather the TP samples of the trajectory that starts at canvas index `base`; offrow = this velocity's row of the
// offset table (kb_tp4(TP) entries, 16-byte aligned).  n = number of valid samples.
template <int TP>
__device__ __forceinline__ void kb_gather_s4(const float2* __restrict__ S4, unsigned int base,
                                             const int4* __restrict__ offrow, float (&f)[TP], float (&m)[TP], int& n) {
    unsigned int cnt = 0u;
#pragma unroll
    for (int q = 0; q < (TP + 3) / 4; ++q) {
        const int4 o = __ldg(offrow + q);
        const int oo[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int t = 4 * q + i;
            if (t < TP) {
                const float2 s = __ldg(S4 + (base + (unsigned int)oo[i]));
                f[t] = s.x;
                m[t] = s.y;
                cnt += __float_as_uint(s.y) >> 31;  // the sign bit of m is the valid flag
            }
        }
    }
    n = (int)cnt;
}

// kept sums of one sample: psi = f |m| (one fused multiply-add), phi = |m| or m^2
template <bool SQ>
__device__ __forceinline__ void kb_accumulate(float f, float m, float& sp, float& sf) {
    sp = __fmaf_rn(f, -m, sp);
    sf = SQ ? __fmaf_rn(m, m, sf) : __fsub_rn(sf, m);
}

// nk = number of kept samples if COUNT, else 1 if anything was kept (sum phi > 0) and 0 if not
template <int TP, bool SQ, bool COUNT>
__device__ __forceinline__ int kb_kept_sums(const float (&f)[TP], const float (&m)[TP], int n, const DevParams& P,
                                            float lo, float hi, float& sp, float& sf) {
    int nk = 0;
    if (!P.sigmag_enable) {
#pragma unroll
        for (int t = 0; t < TP; ++t)
            if (m[t] < 0.0f) kb_accumulate<SQ>(f[t], m[t], sp, sf);
        nk = n;
    } else if (hi < CUDART_INF_F) {
        // an invalid sample (f = +inf) fails f <= hi on its own
#pragma unroll
        for (int t = 0; t < TP; ++t) {
            if (f[t] >= lo && f[t] <= hi) {
                kb_accumulate<SQ>(f[t], m[t], sp, sf);
                if (COUNT) ++nk;
            }
        }
    } else {  // hi = +inf (or NaN: then nothing is kept either way): the validity test is needed
#pragma unroll
        for (int t = 0; t < TP; ++t) {
            if (m[t] < 0.0f && f[t] >= lo && f[t] <= hi) {
                kb_accumulate<SQ>(f[t], m[t], sp, sf);
                if (COUNT) ++nk;
            }
        }
    }
    if (!COUNT && P.sigmag_enable) nk = sf > 0.0f ? 1 : 0;  // every kept sample adds phi > 0
    return nk;
}

// sigma-G filter + kept sums of a gathered trajectory (the search kernels' form of kb_score_lightcurve: the filter
// values come from the canvas instead of 26 divides; invalid samples carry f = +inf, m = 0).
// Returns n_kept (COUNT; 0 = no result) or just non-zero / zero; sp, sf = kept sums.
template <int TP, bool COUNT>
__device__ __forceinline__ int kb_score_s4(const float (&f)[TP], const float (&m)[TP], int n, const DevParams& P,
                                           float* scratch, int stride, float& sp, float& sf) {
    sp = 0.0f;
    sf = 0.0f;
    const int need = P.min_obs > 1 ? P.min_obs : 1;
    if (n < need) return 0;
    float lo = -CUDART_INF_F, hi = CUDART_INF_F;
    if (P.sigmag_enable) {
        float s[TP];
#pragma unroll
        for (int t = 0; t < TP; ++t) s[t] = f[t];
        kb_clip_window<TP>(s, n, P, scratch, stride, lo, hi);
    }
    return P.filter_on ? kb_kept_sums<TP, true, COUNT>(f, m, n, P, lo, hi, sp, sf)
                       : kb_kept_sums<TP, false, COUNT>(f, m, n, P, lo, hi, sp, sf);
}

// 64-bit top-K key: (orderable L', ~velocity index); larger key = better result (L' desc, then vel_idx asc); 0 = empty
__device__ __forceinline__ unsigned int kb_orderable(float f) {
    const unsigned int u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ unsigned long long kb_topk_key(float lh, int v) {
    return ((unsigned long long)kb_orderable(lh) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned)v);
}

// ---------------------------------------------------------------------------------------------
// optional phase timing of kbmod_search (kbmod_search_phase_timing / kbmod_search_phase_ms): an event is recorded
// on the caller's stream after the work of each phase has been enqueued.  No-ops unless timing is switched on.
enum { KB_PHASE_START = -1, KB_PHASE_PLANES = 0, KB_PHASE_BOUND = 1, KB_PHASE_EXACT = 2, KB_PHASE_FINALIZE = 3 };
void kb_phase_mark(int phase, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// host: the geometry-only plan of the pruned search (velocity groups, staging geometry, on-image masks) and the
// device copies of its tables.  Built once per (T, H, W, row band, displacement table); search_pruned.cu
struct PrunedPlan {
    int T = 0, H = 0, W = 0, row_begin = 0, row_end = 0, n_vel = 0, ng = 0, ring_bytes = 0, tiles_x = 0, tiles_y = 0;
    int too_scattered = 0;            // more groups than the workspace layout allows: AUTO falls back to the direct kernel
    double staged = 0.0, evals = 0.0;  // bytes staged / evaluations covered per tile (before off-image skipping)
    double off_image = 0.0;            // share of the (tile, group, epoch) region loads that lie off the image
    double gather_fraction = 1.0;      // shared-memory gathers per nominal evaluation (uniform epochs: one per pixel)
    std::vector<int32_t> gvel;              // [ng][16] velocity index or -1
    std::vector<unsigned char> gtbl;        // [ng] table blocks
    std::vector<unsigned long long> maskx;  // [ng][tiles_x]
    std::vector<unsigned long long> masky;  // [ng][tiles_y]
    std::vector<uint32_t> gfoot;            // [ng]
};
struct PrunedTablesDev {  // device pointers of the uploaded tables
    const int32_t* gvel;
    const unsigned char* gtbl;
    const unsigned long long *maskx, *masky;
    const uint32_t* gfoot;
};
int kb_pruned_plan_build(int T, int H, int W, int row_begin, int row_end, const int32_t* h_dx, const int32_t* h_dy,
                         int n_vel, PrunedPlan* out);
// scratch of the pruned kernels behind the tables: bound planes, survivor queue, scale table, overflow bitmap
size_t kb_pruned_scratch_bytes(int T, int H, int W, int n_rows, int n_vel);
int kb_launch_search_pruned(const float* d_psiphi, const PrunedPlan& plan, const PrunedTablesDev& tb, int TP,
                            const void* d_S4, const S4Geom& G, const int* d_off, const kbmod_search_params* p,
                            const DevParams& P, unsigned long long* d_keys, void* d_scratch, size_t scratch_bytes,
                            unsigned long long* d_stats, cudaStream_t st, int* n_launches);

// S4 canvas and shared kernels (search_common.cu)
int kb_s4_plan(int T, int TP, int H, int W, const int32_t* h_dx, const int32_t* h_dy, int n_vel, S4Geom* G,
               std::vector<int32_t>* off);
size_t kb_s4_bytes(const S4Geom& G, int T);
int kb_launch_s4_build(const float* d_psiphi, int T, int H, int W, const S4Geom& G, int filter_on, void* d_S4,
                       cudaStream_t st);
int kb_launch_finalize(int TP, const unsigned long long* d_keys, const void* d_S4, const S4Geom& G, const int* d_off,
                       int W, int row_begin, int n_rows, const DevParams& P, float* d_lh, float* d_flux, int32_t* d_vel,
                       int32_t* d_nobs, cudaStream_t st);
int kb_launch_unfiltered_lh(int TP, const int32_t* d_vel_idx, const void* d_S4, const S4Geom& G, const int* d_off, int W,
                            int row_begin, int n_rows, int K, int n_vel, int filter_on, float* d_lh_raw, cudaStream_t st);
int kb_write_stats(unsigned long long* d_stats, unsigned long long nominal, unsigned long long launches,
                   unsigned long long algo, unsigned long long evaluated_all, cudaStream_t st);
int kb_launch_search_direct(int TP, const void* d_S4, const S4Geom& G, const int* d_off, const int* d_order, int W,
                            int row_begin, int row_end, int n_vel, const DevParams& P, unsigned long long* d_keys,
                            unsigned long long* d_next_unit, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// launchers (one per .cu file); all return a KBMOD_* status
int kb_launch_prep(const float* d_img, const float* d_var, const uint8_t* d_mask, int T, int H, int W,
                   const float* h_psf, int n_psf, int k, float* d_psiphi, cudaStream_t st);
int kb_launch_eval_trajectories(const float* d_psiphi, int T, int TP, int H, int W, const DevTimes& times,
                                const int32_t* d_x0, const int32_t* d_y0, const float* d_vx, const float* d_vy,
                                int n_traj, const DevParams& P, float* d_psi_lc, float* d_phi_lc,
                                unsigned long long* d_valid, unsigned long long* d_kept, float* d_lh, float* d_flux,
                                cudaStream_t st);
int kb_launch_sigmag_filter(const float* d_psi_lc, const float* d_phi_lc, int n_lc, int T, int TP,
                            const DevParams& P, unsigned long long* d_kept, float* d_lh, float* d_flux,
                            uint8_t* d_pass, unsigned long long* d_n_pass, int32_t* d_survivors, cudaStream_t st);
int kb_launch_coadd(const float* d_img, const uint8_t* d_mask, int T, int TP, int H, int W, const DevTimes& times,
                    const int32_t* d_x0, const int32_t* d_y0, const float* d_vx, const float* d_vy,
                    const unsigned long long* d_epoch_mask, int n_traj, int radius, float* d_mean, float* d_median,
                    const double* thr5, double* d_moments, uint8_t* d_keep, cudaStream_t st);

int kb_launch_stamp_moments(const float* d_stamps, int n, int radius, const double* thr5, double* d_moments,
                            uint8_t* d_pass, cudaStream_t st);
