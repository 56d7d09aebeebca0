// (N2) central-moment stamp filter -- PAPER.md:L141 (s3.3): "we computed the central moments of postage stamps
// ... we required that the x, y, xy, xx, and yy moments be strictly less than 0.5, 0.5, 1.5, 36.5, and 36.5".
// Reading R22: weights w = (I - min I) / sum(I - min I) (uniform for a constant stamp), moments about
// the centre pixel in pixel units, the first three compared by absolute value; a non-finite pixel fails the stamp.
// One warp per stamp: lanes stride over the (2r+1)^2 pixels, minimum and the six sums by warp shuffles.  The sums
// are double precision (the decision precision of this step: 441 x 6 multiply-adds per stamp is nothing).
#include "common.cuh"

namespace {

struct MomentThr {
    double t[5];
};

constexpr int MOM_WARPS = 8;

__global__ void __launch_bounds__(32 * MOM_WARPS)
stamp_moments_kernel(const float* __restrict__ stamps, int n, int radius, const __grid_constant__ MomentThr thr,
                     double* __restrict__ moments, uint8_t* __restrict__ pass) {
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * MOM_WARPS + (threadIdx.x >> 5);
    if (i >= n) return;
    const int S = 2 * radius + 1, N = S * S;
    const float* I = stamps + (size_t)i * N;
    float mn = CUDART_INF_F;
    bool finite = true;
    for (int k = lane; k < N; k += 32) {
        const float x = __ldg(I + k);
        finite = finite && (fabsf(x) < CUDART_INF_F);  // false for NaN, too
        mn = fminf(mn, x);
    }
    for (int d = 16; d > 0; d >>= 1) mn = fminf(mn, __shfl_xor_sync(0xFFFFFFFFu, mn, d));
    finite = __all_sync(0xFFFFFFFFu, finite);
    double s0 = 0.0, sx = 0.0, sy = 0.0, sxy = 0.0, sxx = 0.0, syy = 0.0;
    if (finite) {
        for (int k = lane; k < N; k += 32) {
            const int v = k / S - radius, u = k % S - radius;
            const double w = (double)__ldg(I + k) - (double)mn;
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
    if (lane != 0) return;
    double m[5];
    bool keep = false;
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
    if (moments)
        for (int k = 0; k < 5; ++k) moments[(size_t)i * 5 + k] = m[k];
    if (pass) pass[i] = keep ? 1 : 0;
}

}  // namespace

int kb_launch_stamp_moments(const float* d_stamps, int n, int radius, const double* thr5, double* d_moments,
                            uint8_t* d_pass, cudaStream_t st) {
    MomentThr thr;
    for (int k = 0; k < 5; ++k) thr.t[k] = thr5[k];
    stamp_moments_kernel<<<(n + MOM_WARPS - 1) / MOM_WARPS, 32 * MOM_WARPS, 0, st>>>(d_stamps, n, radius, thr, d_moments,
                                                                                      d_pass);
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}
