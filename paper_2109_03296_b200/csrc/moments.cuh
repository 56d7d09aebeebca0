// Central moments of one stamp by one warp (s3.3; reading R22) -- shared by the stand-alone
// stamp_moments_kernel and by coadd_kernel's fused output, so that both produce the same bits.
// Weights w = (I - min I) / sum(I - min I) (uniform for a constant stamp), moments about the centre pixel in pixel
// units; a non-finite pixel fails the stamp (NaN moments).  Lanes stride over the (2r+1)^2 pixels, minimum and the six
// sums by warp shuffles, sums in double (the decision precision of this step).
#pragma once
#include "common.cuh"

struct MomentThr {
    double t[5];
};

// all 32 lanes must call; `I` may point to global or shared memory.  Results are valid in lane 0.
__device__ __forceinline__ void kb_moments_warp(const float* I, int radius, const MomentThr& thr, double (&m)[5],
                                                bool& keep) {
    const int lane = threadIdx.x & 31;
    const int S = 2 * radius + 1, N = S * S;
    float mn = CUDART_INF_F;
    bool finite = true;
    for (int k = lane; k < N; k += 32) {
        const float x = I[k];
        finite = finite && (fabsf(x) < CUDART_INF_F);  // false for NaN, too
        mn = fminf(mn, x);
    }
    for (int d = 16; d > 0; d >>= 1) mn = fminf(mn, __shfl_xor_sync(0xFFFFFFFFu, mn, d));
    finite = __all_sync(0xFFFFFFFFu, finite);
    double s0 = 0.0, sx = 0.0, sy = 0.0, sxy = 0.0, sxx = 0.0, syy = 0.0;
    if (finite) {
        for (int k = lane; k < N; k += 32) {
            const int v = k / S - radius, u = k % S - radius;
            const double w = (double)I[k] - (double)mn;
            s0 += w;
            sx += u * w;
            sy += v * w;
            sxy += (double)(u * v) * w;
            sxx += (double)(u * u) * w;
            syy += (double)(v * v) * w;
        }
        for (int d = 16; d > 0; d >>= 1) {
            s0 += __shfl_xor_sync(0xFFFFFFFFu, s0, d);
            sx += __shfl_xor_sync(0xFFFFFFFFu, sx, d);
            sy += __shfl_xor_sync(0xFFFFFFFFu, sy, d);
            sxy += __shfl_xor_sync(0xFFFFFFFFu, sxy, d);
            sxx += __shfl_xor_sync(0xFFFFFFFFu, sxx, d);
            syy += __shfl_xor_sync(0xFFFFFFFFu, syy, d);
        }
    }
    keep = false;
    if (!finite) {
        for (int k = 0; k < 5; ++k) m[k] = CUDART_NAN;
    } else {
        if (s0 > 0.0) {
            m[0] = sx / s0; m[1] = sy / s0; m[2] = sxy / s0; m[3] = sxx / s0; m[4] = syy / s0;
        } else {  // a constant stamp: uniform weights, second moments r (r + 1) / 3
            m[0] = m[1] = m[2] = 0.0;
            m[3] = m[4] = (double)radius * (double)(radius + 1) / 3.0;
        }
        keep = fabs(m[0]) < thr.t[0] && fabs(m[1]) < thr.t[1] && fabs(m[2]) < thr.t[2] && m[3] < thr.t[3] && m[4] < thr.t[4];
    }
}
