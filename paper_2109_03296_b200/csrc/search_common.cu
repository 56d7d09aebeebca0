// Pieces both search kernels share (common.cuh "S4"): the padded float4 working copy of the psi/phi stack, the
// per-velocity offset table into it, and the kernel that turns per-pixel top-K keys into the four output arrays.
// PAPER.md:L79-L81 (s3): the search sums "previously-calculated likelihoods" along a trajectory by "pointer
// arithmetic"; here every sample is one 16-byte load at base(x0, y0) + off[v][t], with the off-chip rule
// (reading R8: such epochs contribute nothing) carried by the padding instead of a bounds test.
#include <algorithm>
#include <vector>

#include "common.cuh"

namespace {

// one thread per canvas pixel of planes 0..T (plane T is the all-invalid plane padding epochs point into)
__global__ void __launch_bounds__(256)
s4_build_kernel(const float2* __restrict__ psiphi, float2* __restrict__ S4, int T, int H, int W,
                const __grid_constant__ S4Geom G, int filter_on) {
    const unsigned int xp = blockIdx.x * 256u + threadIdx.x;
    if (xp >= (unsigned int)G.Wp) return;
    const int yp = blockIdx.y, t = blockIdx.z;
    const int x = (int)xp - G.pxn, y = yp - G.pyn;
    float2 o = make_float2(CUDART_INF_F, 0.0f);  // (f, m): common.cuh "canvas"
    if (t < T && x >= 0 && x < W && y >= 0 && y < H) {
        const float2 s = __ldg(psiphi + ((size_t)t * H + y) * W + x);
        if (s.y > 0.0f)  // reading R21: a sample is valid iff phi > 0 (prep writes (0, 0) for invalid pixels)
            o = make_float2(kb_filter_value(s.x, s.y, filter_on), filter_on ? -__fsqrt_rn(s.y) : -s.y);
    }
    S4[(size_t)t * G.plane + (size_t)yp * G.Wp + xp] = o;
}

// keys -> output arrays.  One thread per (band pixel, slot); a filled slot is re-evaluated to get flux and n_obs
// (the key carries L' and the velocity index only).
constexpr int FIN_THREADS = 128;

template <int TP>
__global__ void __launch_bounds__(FIN_THREADS)
finalize_kernel(const unsigned long long* __restrict__ keys, const float2* __restrict__ S4,
                const __grid_constant__ S4Geom G, const int* __restrict__ off, int W, int row_begin, int n_rows,
                const __grid_constant__ DevParams P, float* __restrict__ out_lh, float* __restrict__ out_flux,
                int32_t* __restrict__ out_vel, int32_t* __restrict__ out_nobs) {
    extern __shared__ float scratch_all[];
    const size_t i = (size_t)blockIdx.x * FIN_THREADS + threadIdx.x;
    const size_t total = (size_t)n_rows * W * P.K;
    if (i >= total) return;
    const unsigned long long key = keys[i];
    float lh = -CUDART_INF_F, flux = 0.0f;
    int vel = -1, nobs = 0;
    if (key != 0ull) {
        vel = (int)(0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull));
        const int pixlin = (int)(i / P.K);
        const int yb = pixlin / W, x0 = pixlin - yb * W;
        const unsigned int base = (unsigned int)(yb + row_begin + G.pyn) * (unsigned int)G.Wp + (unsigned int)(x0 + G.pxn);
        float f[TP], m[TP], sp, sf;
        int n;
        kb_gather_s4<TP>(S4, base, reinterpret_cast<const int4*>(off + (size_t)vel * kb_tp4(TP)), f, m, n);
        nobs = kb_score_s4<TP, true>(f, m, n, P, scratch_all + threadIdx.x, FIN_THREADS, sp, sf);
        lh = kb_lh_of(sp, sf);
        flux = kb_flux_of(sp, sf);
    }
    out_lh[i] = lh;
    out_flux[i] = flux;
    out_vel[i] = vel;
    out_nobs[i] = nobs;
}

// unfiltered sum-LH of every result slot: sum over ALL valid epochs, no clip, no threshold
template <int TP>
__global__ void __launch_bounds__(FIN_THREADS)
unfiltered_lh_kernel(const int32_t* __restrict__ vel_idx, const float2* __restrict__ S4, const __grid_constant__ S4Geom G,
                     const int* __restrict__ off, int W, int row_begin, int n_rows, int K, int n_vel, int filter_on,
                     float* __restrict__ out_lh) {
    const size_t i = (size_t)blockIdx.x * FIN_THREADS + threadIdx.x;
    const size_t total = (size_t)n_rows * W * K;
    if (i >= total) return;
    const int vel = vel_idx[i];
    float lh = -CUDART_INF_F;
    if (vel >= 0 && vel < n_vel) {
        const int pixlin = (int)(i / K);
        const int yb = pixlin / W, x0 = pixlin - yb * W;
        const unsigned int base = (unsigned int)(yb + row_begin + G.pyn) * (unsigned int)G.Wp + (unsigned int)(x0 + G.pxn);
        float f[TP], m[TP];
        int n;
        kb_gather_s4<TP>(S4, base, reinterpret_cast<const int4*>(off + (size_t)vel * kb_tp4(TP)), f, m, n);
        float sp = 0.0f, sf = 0.0f;
#pragma unroll
        for (int t = 0; t < TP; ++t) {
            if (m[t] < 0.0f) {
                if (filter_on) kb_accumulate<true>(f[t], m[t], sp, sf);
                else kb_accumulate<false>(f[t], m[t], sp, sf);
            }
        }
        if (n > 0) lh = kb_lh_of(sp, sf);
    }
    out_lh[i] = lh;
}

// counters of kbmod_search_stats: written on the stream from kernel arguments (no host buffer outlives the call)
__global__ void write_stats_kernel(unsigned long long* s, unsigned long long nominal, unsigned long long launches,
                                   unsigned long long algo, unsigned long long evaluated_all) {
    if (evaluated_all) s[0] = evaluated_all;
    s[1] = nominal;
    s[2] = launches;
    s[3] = algo;
}

}  // namespace

int kb_write_stats(unsigned long long* d_stats, unsigned long long nominal, unsigned long long launches,
                   unsigned long long algo, unsigned long long evaluated_all, cudaStream_t st) {
    write_stats_kernel<<<1, 1, 0, st>>>(d_stats, nominal, launches, algo, evaluated_all);
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}

// ---------------------------------------------------------------------------------------------
// host: canvas geometry and offset table from the displacement table (a2).  A displacement beyond the image size
// can never land on the image, wherever exactly it points: it is clamped to the image size, which the padding
// covers, so the offset stays small and the sample reads "invalid".
int kb_s4_plan(int T, int TP, int H, int W, const int32_t* h_dx, const int32_t* h_dy, int n_vel, S4Geom* G,
               std::vector<int32_t>* off) {
    int pxn = 0, pxp = 0, pyn = 0, pyp = 0;
    for (size_t i = 0; i < (size_t)n_vel * T; ++i) {
        const int dx = std::max(-W, std::min(W, h_dx[i])), dy = std::max(-H, std::min(H, h_dy[i]));
        pxn = std::max(pxn, -dx); pxp = std::max(pxp, dx);
        pyn = std::max(pyn, -dy); pyp = std::max(pyp, dy);
    }
    G->pxn = pxn; G->pyn = pyn;
    G->Wp = W + pxn + pxp; G->Hp = H + pyn + pyp;
    const double plane = (double)G->Wp * (double)G->Hp;
    KB_REQUIRE(plane * (T + 1) < 4294967296.0, KBMOD_ERR_UNSUPPORTED,
               "search canvas of (T + 1) x %d x %d pixels exceeds 2^32 (displacements up to %d, %d px pad the %d x %d image)",
               G->Wp, G->Hp, std::max(pxn, pxp), std::max(pyn, pyp), W, H);
    G->plane = (unsigned int)plane;
    if (off) {
        const int TP4 = kb_tp4(TP);
        off->assign((size_t)n_vel * TP4, 0);
        for (int v = 0; v < n_vel; ++v)
            for (int t = 0; t < TP4; ++t) {
                long long o;
                if (t < T) {
                    const int dx = std::max(-W, std::min(W, h_dx[(size_t)v * T + t]));
                    const int dy = std::max(-H, std::min(H, h_dy[(size_t)v * T + t]));
                    o = (long long)t * G->plane + (long long)dy * G->Wp + dx;
                } else {
                    o = (long long)T * G->plane;  // the all-invalid plane
                }
                // base + o is evaluated modulo 2^32 on the device; the true sum lies in [0, 2^32) by construction
                (*off)[(size_t)v * TP4 + t] = (int32_t)(uint32_t)(unsigned long long)o;
            }
    }
    return KBMOD_OK;
}

size_t kb_s4_bytes(const S4Geom& G, int T) { return (size_t)G.plane * (size_t)(T + 1) * sizeof(float2); }

int kb_launch_s4_build(const float* d_psiphi, int T, int H, int W, const S4Geom& G, int filter_on, void* d_S4,
                       cudaStream_t st) {
    const dim3 grid((unsigned)((G.Wp + 255) / 256), (unsigned)G.Hp, (unsigned)(T + 1));
    KB_REQUIRE(G.Hp <= 65535 && T + 1 <= 65535, KBMOD_ERR_UNSUPPORTED, "canvas of %d rows exceeds the grid limit", G.Hp);
    s4_build_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const float2*>(d_psiphi), reinterpret_cast<float2*>(d_S4), T, H,
                                          W, G, filter_on);
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}

int kb_launch_finalize(int TPv, const unsigned long long* d_keys, const void* d_S4, const S4Geom& G, const int* d_off,
                       int W, int row_begin, int n_rows, const DevParams& P, float* d_lh, float* d_flux, int32_t* d_vel,
                       int32_t* d_nobs, cudaStream_t st) {
    const size_t total = (size_t)n_rows * W * P.K;
    if (total == 0) return KBMOD_OK;
    KB_DISPATCH_TP(TPv, {
        const size_t smem = (size_t)TP * FIN_THREADS * sizeof(float);
        finalize_kernel<TP><<<(unsigned)((total + FIN_THREADS - 1) / FIN_THREADS), FIN_THREADS, smem, st>>>(
            d_keys, reinterpret_cast<const float2*>(d_S4), G, d_off, W, row_begin, n_rows, P, d_lh, d_flux, d_vel, d_nobs);
    });
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}

int kb_launch_unfiltered_lh(int TPv, const int32_t* d_vel_idx, const void* d_S4, const S4Geom& G, const int* d_off, int W,
                            int row_begin, int n_rows, int K, int n_vel, int filter_on, float* d_lh_raw, cudaStream_t st) {
    const size_t total = (size_t)n_rows * W * K;
    if (total == 0) return KBMOD_OK;
    KB_DISPATCH_TP(TPv, {
        unfiltered_lh_kernel<TP><<<(unsigned)((total + FIN_THREADS - 1) / FIN_THREADS), FIN_THREADS, 0, st>>>(
            d_vel_idx, reinterpret_cast<const float2*>(d_S4), G, d_off, W, row_begin, n_rows, K, n_vel, filter_on, d_lh_raw);
    });
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}
