// (a3)-(a5) direct search: one thread per start pixel walks every velocity, gathers the T samples
// through L1 (a warp is 32 consecutive x0, so each epoch is one 256-byte row segment), runs the
// sigma-G filter on the register-resident lightcurve and keeps its pixel's top-K.
// PAPER.md:L79-L81 (s3), L93-L117 (s3.1), L127-L137 (s3.2); steps 1-4 of kbmod_search in
// include/kbmod_b200.h.  This is the evaluator for every trajectory when no threshold prunes
// (min_lh = -inf) and the reference implementation the pruned kernel must agree with.
#include "common.cuh"

namespace {

constexpr int SD_BX = 32, SD_BY = 4;  // block = 4 warps, each a 32-pixel row segment

template <int TP>
__global__ void __launch_bounds__(SD_BX* SD_BY)
search_direct_kernel(const float2* __restrict__ psiphi, int H, int W, const DispEntry* __restrict__ tab, int n_vel,
                     const __grid_constant__ DevParams P, float* __restrict__ out_lh, float* __restrict__ out_flux,
                     int32_t* __restrict__ out_vel, int32_t* __restrict__ out_nobs) {
    extern __shared__ float scratch_all[];  // [TP][threads]
    const int tid = threadIdx.y * SD_BX + threadIdx.x;
    float* scratch = scratch_all + tid;
    constexpr int stride = SD_BX * SD_BY;

    const int x0 = blockIdx.x * SD_BX + threadIdx.x;
    const int y0 = blockIdx.y * SD_BY + threadIdx.y;
    if (x0 >= W || y0 >= H) return;
    const int pix = y0 * W + x0;
    const int K = P.K;
    const size_t base = (size_t)pix * K;
    for (int k = 0; k < K; ++k) {
        out_lh[base + k] = -CUDART_INF_F;
        out_flux[base + k] = 0.0f;
        out_vel[base + k] = -1;
        out_nobs[base + k] = 0;
    }
    int cnt = 0;
    float kth = -CUDART_INF_F;  // L' of slot K-1 once the list is full

    const unsigned warp_mask = __activemask();  // lanes past the right edge have left
#pragma unroll 1
    for (int v = 0; v < n_vel; ++v) {
        __syncwarp(warp_mask);  // re-converge after the divergent top-K insertion of the previous velocity
        const DispEntry* row = tab + (size_t)v * TP;
        float psi[TP], phi[TP];
#pragma unroll
        for (int t = 0; t < TP; ++t) {
            const DispEntry e = row[t];  // warp-uniform address
            const int x = x0 + e.dx, y = y0 + e.dy;
            float2 s = make_float2(0.0f, 0.0f);
            if ((unsigned)x < (unsigned)W && (unsigned)y < (unsigned)H) s = __ldg(psiphi + (pix + e.off));
            const bool ok = s.y > 0.0f;  // invalid pixels are stored as (0, 0)
            psi[t] = ok ? s.x : 0.0f;
            phi[t] = ok ? s.y : 0.0f;
        }
        float lh, flux;
        unsigned long long kept;
        const int nk = kb_score_lightcurve<TP>(psi, phi, P, scratch, stride, lh, flux, kept);
        if (nk == 0 || !(lh >= P.min_lh)) continue;
        if (cnt == K && !(lh > kth)) continue;
        // insert: velocities arrive in ascending index, so strict '>' keeps the lower index first
        int pos = cnt < K ? cnt : K - 1;
        while (pos > 0 && lh > out_lh[base + pos - 1]) {
            out_lh[base + pos] = out_lh[base + pos - 1];
            out_flux[base + pos] = out_flux[base + pos - 1];
            out_vel[base + pos] = out_vel[base + pos - 1];
            out_nobs[base + pos] = out_nobs[base + pos - 1];
            --pos;
        }
        out_lh[base + pos] = lh;
        out_flux[base + pos] = flux;
        out_vel[base + pos] = v;
        out_nobs[base + pos] = nk;
        if (cnt < K) ++cnt;
        if (cnt == K) kth = out_lh[base + K - 1];
    }
}

}  // namespace

int kb_launch_search_direct(const float* d_psiphi, int T, int TPv, int H, int W, const DispEntry* d_tab, int n_vel,
                            const DevParams& P, float* d_lh, float* d_flux, int32_t* d_vel, int32_t* d_nobs,
                            cudaStream_t st) {
    (void)T;
    const dim3 block(SD_BX, SD_BY);
    const dim3 grid((W + SD_BX - 1) / SD_BX, (H + SD_BY - 1) / SD_BY);
    KB_DISPATCH_TP(TPv, {
        const size_t smem = (size_t)TP * SD_BX * SD_BY * sizeof(float);
        search_direct_kernel<TP><<<grid, block, smem, st>>>(reinterpret_cast<const float2*>(d_psiphi), H, W, d_tab,
                                                            n_vel, P, d_lh, d_flux, d_vel, d_nobs);
    });
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}
