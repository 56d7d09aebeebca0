// (N2) central-moment stamp filter -- PAPER.md:L141 (s3.3): "we computed the central moments of postage stamps
// ... we required that the x, y, xy, xx, and yy moments be strictly less than 0.5, 0.5, 1.5, 36.5, and 36.5".
// Reading R22: weights w = (I - min I) / sum(I - min I) (uniform for a constant stamp), moments about
// the centre pixel in pixel units, the first three compared by absolute value; a non-finite pixel fails the stamp.
// One warp per stamp: lanes stride over the (2r+1)^2 pixels, minimum and the six sums by warp shuffles.  The sums
// are double precision (the decision precision of this step: 441 x 6 multiply-adds per stamp is nothing).
#include "moments.cuh"

namespace {

constexpr int MOM_WARPS = 8;

__global__ void __launch_bounds__(32 * MOM_WARPS)
stamp_moments_kernel(const float* __restrict__ stamps, int n, int radius, const __grid_constant__ MomentThr thr,
                     double* __restrict__ moments, uint8_t* __restrict__ pass) {
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * MOM_WARPS + (threadIdx.x >> 5);
    if (i >= n) return;
    const int S = 2 * radius + 1;
    double m[5];
    bool keep;
    kb_moments_warp(stamps + (size_t)i * S * S, radius, thr, m, keep);
    if (lane != 0) return;
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
