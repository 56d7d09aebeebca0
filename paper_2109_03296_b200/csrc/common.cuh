// Internal declarations shared by the kernels of libkbmod_b200.so.  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>
#include <stdio.h>

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
    int sigmag_enable, filter_on, min_obs, K, T;
    float coeff, n_sigma, min_lh;
    // nearest-rank percentile index ceil(q n / 100) - 1 clamped to [0, n-1], for n = 0..64
    // ("selecting the 25th and 75th percentile values ... from the data"; reading R10)
    unsigned char rk_lo[KBMOD_MAX_T + 1], rk_md[KBMOD_MAX_T + 1], rk_hi[KBMOD_MAX_T + 1];
};
struct DevTimes {
    double dt[KBMOD_MAX_T];  // times[t] - times[0]
};

int kb_make_dev_params(const kbmod_search_params* p, int T, DevParams* out);  // validates
int kb_padded_T(int T);  // smallest instantiated network size >= T, or -1

// One entry per (velocity, epoch) of the displacement table as the search kernels read it.
struct __align__(8) DispEntry {
    int32_t off;    // t*H*W + dy*W + dx : added to y0*W + x0 it indexes the [T][H][W] stack
    int16_t dx, dy; // for the on-image test; dx = -32768 marks a padding epoch (t >= T)
};

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

// device: sigma-G filter + score of one lightcurve held in registers (steps 2-3 of kbmod_search;
// PAPER.md:L95-L117 Eq. 1-5).  Epoch t is valid iff phi[t] > 0.
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
            // IEEE float32, correctly rounded: the precision the keep/drop decision is taken in
            // invalid epochs divide 1 by 1: a zero operand would send the whole warp down the slow path of the divide
            // (an invalid epoch divides by zero and the result is discarded: guarding the operands instead was
            // measured 2-3 % slower once the warps stay converged)
            const float den = P.filter_on ? __fsqrt_rn(phi[t]) : phi[t];
            f[t] = (phi[t] > 0.0f) ? __fdiv_rn(psi[t], den) : CUDART_INF_F;
            s[t] = f[t];
        }
        SortNet<TP>::sort(s);  // invalid epochs (+inf) end up behind the n valid ones
#pragma unroll
        for (int t = 0; t < TP; ++t) scratch[t * stride] = s[t];
        const float p_lo = scratch[P.rk_lo[n] * stride];
        const float p_50 = scratch[P.rk_md[n] * stride];
        const float p_hi = scratch[P.rk_hi[n] * stride];
        const float d = __fsub_rn(p_hi, p_lo);      // Eq. 5: sigma_G = C (x_j - x_i)
        const float sg = __fmul_rn(P.coeff, d);
        const float w = __fmul_rn(P.n_sigma, sg);   // L117: +- n sigma_G about the median
        lo = __fsub_rn(p_50, w);
        hi = __fadd_rn(p_50, w);
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
    lh = sp / sqrtf(sf);  // L79: nu = Psi_coadd / sqrt(Phi_coadd), recomputed from the survivors (L123)
    flux = sp / sf;
    return nk;
}

// ---------------------------------------------------------------------------------------------
// optional phase timing of kbmod_search (kbmod_search_phase_timing / kbmod_search_phase_ms): an event is recorded
// on the caller's stream after the work of each phase has been enqueued.  No-ops unless timing is switched on.
enum { KB_PHASE_START = -1, KB_PHASE_PLANES = 0, KB_PHASE_BOUND = 1, KB_PHASE_EXACT = 2, KB_PHASE_FINALIZE = 3 };
void kb_phase_mark(int phase, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// launchers (one per .cu file); all return a KBMOD_* status
int kb_launch_prep(const float* d_img, const float* d_var, const uint8_t* d_mask, int T, int H, int W,
                   const float* h_psf, int n_psf, int k, float* d_psiphi, cudaStream_t st);
int kb_launch_search_direct(const float* d_psiphi, int T, int TP, int H, int W, const DispEntry* d_tab, int n_vel,
                            const DevParams& P, float* d_lh, float* d_flux, int32_t* d_vel, int32_t* d_nobs,
                            cudaStream_t st);
int kb_launch_eval_trajectories(const float* d_psiphi, int T, int TP, int H, int W, const DevTimes& times,
                                const int32_t* d_x0, const int32_t* d_y0, const float* d_vx, const float* d_vy,
                                int n_traj, const DevParams& P, float* d_psi_lc, float* d_phi_lc,
                                unsigned long long* d_valid, unsigned long long* d_kept, float* d_lh, float* d_flux,
                                cudaStream_t st);
int kb_launch_sigmag_filter(const float* d_psi_lc, const float* d_phi_lc, int n_lc, int T, int TP,
                            const DevParams& P, unsigned long long* d_kept, float* d_lh, float* d_flux,
                            cudaStream_t st);
int kb_launch_coadd(const float* d_img, const uint8_t* d_mask, int T, int TP, int H, int W, const DevTimes& times,
                    const int32_t* d_x0, const int32_t* d_y0, const float* d_vx, const float* d_vy,
                    const unsigned long long* d_epoch_mask, int n_traj, int radius, float* d_mean, float* d_median,
                    cudaStream_t st);

int kb_launch_stamp_moments(const float* d_stamps, int n, int radius, const double* thr5, double* d_moments,
                            uint8_t* d_pass, cudaStream_t st);

// pruned search (search_pruned.cu).  h_dx, h_dy: [n_vel][T] displacement table (a2).  plan_only: run the host
// planner only and fill plan_stats = {fraction of velocity groups that cannot be staged, staged bytes per evaluation}.
size_t kb_pruned_workspace_bytes(int T, int H, int W, int n_vel, int K);
int kb_launch_search_pruned(const float* d_psiphi, int T, int TP, int H, int W, const DispEntry* d_tab,
                            const int32_t* h_dx, const int32_t* h_dy, int n_vel, const kbmod_search_params* p,
                            const DevParams& P, float* d_lh, float* d_flux, int32_t* d_vel, int32_t* d_nobs,
                            void* d_ws, size_t ws_bytes, unsigned long long* d_stats, cudaStream_t st, int plan_only,
                            double* plan_stats, int* n_launches);
