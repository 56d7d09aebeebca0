// (a6) coadded stamps -- PAPER.md:L141 (s3.3): "computing the median pixel value for each pixel
// along the trajectory"; mean is the earlier variant; 21x21 (L145, L175); reading R17.
// One block per trajectory, one thread per stamp pixel: for each epoch the block reads a
// (2r+1)-wide row segment per stamp row (coalesced within the row), the T samples of a pixel
// stay in registers, and the median comes from the same compare-exchange network as sigma-G
// (with two-sided +-inf padding so that its position is fixed; see below).  Optionally the block goes on to the step
// behind the coadd (L141: "we computed the central moments of postage stamps ..."): the medians are parked in shared
// memory and one warp computes the five moments and the keep flag with the same device function as
// kbmod_stamp_moments -- no second pass over the stamps in global memory.
#include "moments.cuh"

// Blocks of 448 threads per SM the kernel is compiled for.  It is bound by the latency of its scattered 84-byte row
// reads, so residency beats registers: 2 / 3 / 4 blocks per SM (50 / 40 / 32 registers, the last two with a few spilled
// words) take 6.7 / 4.9 / 4.3 ms for 10^5 trajectories x 26 epochs with the moment filter.
#ifndef KB_COADD_BLOCKS
#define KB_COADD_BLOCKS 4
#endif
namespace {

template <int TP>
__global__ void __launch_bounds__(448, KB_COADD_BLOCKS) coadd_kernel(const float* __restrict__ img, const uint8_t* __restrict__ mask, int T, int H, int W,
                             const __grid_constant__ DevTimes times, const int32_t* __restrict__ x0s,
                             const int32_t* __restrict__ y0s, const float* __restrict__ vxs,
                             const float* __restrict__ vys, const unsigned long long* __restrict__ epoch_mask,
                             int radius, float* __restrict__ mean_out, float* __restrict__ median_out, int want_moments,
                             const __grid_constant__ MomentThr thr, double* __restrict__ moments_out,
                             uint8_t* __restrict__ keep_out) {
    __shared__ int sdx[KBMOD_MAX_T], sdy[KBMOD_MAX_T];
    __shared__ float smed[(2 * KBMOD_MAX_STAMP_RADIUS + 1) * (2 * KBMOD_MAX_STAMP_RADIUS + 1)];
    const int i = blockIdx.x;
    const int S = 2 * radius + 1;
    const int x0 = x0s[i], y0 = y0s[i];
    if (threadIdx.x < T) {
        sdx[threadIdx.x] = kb_displacement(vxs[i], times.dt[threadIdx.x]);
        sdy[threadIdx.x] = kb_displacement(vys[i], times.dt[threadIdx.x]);
    }
    __syncthreads();
    const unsigned long long sel = epoch_mask ? epoch_mask[i] : ~0ull;
    const size_t plane = (size_t)H * W;
    for (int p = threadIdx.x; p < S * S; p += blockDim.x) {
    const int v = p / S - radius, u = p % S - radius;

    float vals[TP];
    float sum = 0.0f;
    int m = 0;
    unsigned long long got = 0ull;
#pragma unroll
    for (int t = 0; t < TP; ++t) {
        vals[t] = CUDART_INF_F;
        if (t < T && ((sel >> t) & 1ull)) {
            const int x = x0 + sdx[t] + u, y = y0 + sdy[t] + v;
            if (x >= 0 && x < W && y >= 0 && y < H) {
                const size_t q = t * plane + (size_t)y * W + x;
                const float a = __ldg(img + q);
                if ((!mask || __ldg(mask + q) == 0) && isfinite(a)) {
                    vals[t] = a;
                    sum += a;
                    ++m;
                    got |= 1ull << t;
                }
            }
        }
    }
    float mean = 0.0f, med = 0.0f;
    if (m > 0) {
        mean = sum / (float)m;
        // Median without a data-dependent index: of the TP - m skipped slots the first
        // floor((TP-m)/2) become -inf and the rest +inf, so after the sort the m samples sit in
        // the middle and the median is at fixed positions that depend only on the parity of m.
        const int n_low = (TP - m) >> 1;
        int seen = 0;
#pragma unroll
        for (int t = 0; t < TP; ++t) {
            if (!((got >> t) & 1ull)) {
                vals[t] = (seen < n_low) ? -CUDART_INF_F : CUDART_INF_F;
                ++seen;
            }
        }
        SortNet<TP>::sort(vals);
        constexpr int c_even_a = (TP & 1) ? (TP - 3) / 2 : TP / 2 - 1;  // m even: two middles
        constexpr int c_even_b = (TP & 1) ? (TP - 1) / 2 : TP / 2;
        constexpr int c_odd = (TP & 1) ? (TP - 1) / 2 : TP / 2 - 1;     // m odd: the middle
        med = (m & 1) ? vals[c_odd] : 0.5f * (vals[c_even_a] + vals[c_even_b]);
    }
    const size_t o = (size_t)i * S * S + p;
    if (mean_out) mean_out[o] = mean;
    if (median_out) median_out[o] = med;
    if (want_moments) smed[p] = med;
    }
    if (want_moments) {  // block-uniform
        __syncthreads();
        if (threadIdx.x < 32) {
            double m[5];
            bool keep;
            kb_moments_warp(smed, radius, thr, m, keep);
            if (threadIdx.x == 0) {
                if (moments_out)
                    for (int k = 0; k < 5; ++k) moments_out[(size_t)i * 5 + k] = m[k];
                if (keep_out) keep_out[i] = keep ? 1 : 0;
            }
        }
    }
}

}  // namespace

int kb_launch_coadd(const float* d_img, const uint8_t* d_mask, int T, int TPv, int H, int W, const DevTimes& times,
                    const int32_t* d_x0, const int32_t* d_y0, const float* d_vx, const float* d_vy,
                    const unsigned long long* d_epoch_mask, int n_traj, int radius, float* d_mean, float* d_median,
                    const double* thr5, double* d_moments, uint8_t* d_keep, cudaStream_t st) {
    MomentThr thr;
    for (int k = 0; k < 5; ++k) thr.t[k] = thr5 ? thr5[k] : 0.0;
    const int want_moments = (d_moments || d_keep) ? 1 : 0;
    const int S = 2 * radius + 1;
    int threads = ((S * S + 31) / 32) * 32;  // one stamp pixel per thread up to 21x21, a loop above that
    if (threads < 64) threads = 64;          // the first T threads compute the displacements
    if (threads > 448) threads = 256;
    KB_DISPATCH_TP(TPv, {
        coadd_kernel<TP><<<n_traj, threads, 0, st>>>(d_img, d_mask, T, H, W, times, d_x0, d_y0, d_vx, d_vy,
                                                        d_epoch_mask, radius, d_mean, d_median, want_moments, thr,
                                                        d_moments, d_keep);
    });
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}
