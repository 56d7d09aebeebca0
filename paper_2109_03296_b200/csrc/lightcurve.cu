// Single-trajectory variant (s4.1) and the sigma-G post-filter on given lightcurves
// (s3.1; BASELINE configs[4]).  One thread per trajectory / lightcurve; the filter is
// the same device function the search kernels use (common.cuh: kb_score_lightcurve).
#include <algorithm>
#include <mutex>

#include "common.cuh"

namespace {

constexpr int LC_THREADS = 128;

template <int TP>
__global__ void __launch_bounds__(LC_THREADS)
eval_trajectories_kernel(const float2* __restrict__ psiphi, int T, int H, int W, const __grid_constant__ DevTimes times,
                         const int32_t* __restrict__ x0s, const int32_t* __restrict__ y0s,
                         const float* __restrict__ vxs, const float* __restrict__ vys, int n_traj,
                         const __grid_constant__ DevParams P, float* __restrict__ psi_lc, float* __restrict__ phi_lc,
                         unsigned long long* __restrict__ valid_out, unsigned long long* __restrict__ kept_out,
                         float* __restrict__ lh_out, float* __restrict__ flux_out) {
    extern __shared__ float scratch_all[];
    float* scratch = scratch_all + threadIdx.x;
    const int i = blockIdx.x * LC_THREADS + threadIdx.x;
    if (i >= n_traj) return;
    const int x0 = x0s[i], y0 = y0s[i];
    const float vx = vxs[i], vy = vys[i];
    const size_t plane = (size_t)H * W;
    float psi[TP], phi[TP];
    unsigned long long valid = 0ull;
#pragma unroll
    for (int t = 0; t < TP; ++t) {
        psi[t] = 0.0f;
        phi[t] = 0.0f;
        if (t < T) {
            const int x = x0 + kb_displacement(vx, times.dt[t]);
            const int y = y0 + kb_displacement(vy, times.dt[t]);
            if (x >= 0 && x < W && y >= 0 && y < H) {
                const float2 s = __ldg(psiphi + t * plane + (size_t)y * W + x);
                if (s.y > 0.0f) {
                    psi[t] = s.x;
                    phi[t] = s.y;
                    valid |= 1ull << t;
                }
            }
        }
    }
    float lh, flux;
    unsigned long long kept;
    kb_score_lightcurve<TP>(psi, phi, P, scratch, LC_THREADS, lh, flux, kept);
    if (psi_lc)
#pragma unroll
        for (int t = 0; t < TP; ++t)
            if (t < T) psi_lc[(size_t)i * T + t] = psi[t];
    if (phi_lc)
#pragma unroll
        for (int t = 0; t < TP; ++t)
            if (t < T) phi_lc[(size_t)i * T + t] = phi[t];
    if (valid_out) valid_out[i] = valid;
    if (kept_out) kept_out[i] = kept;
    if (lh_out) lh_out[i] = lh;
    if (flux_out) flux_out[i] = flux;
}

template <int TP>
__global__ void __launch_bounds__(LC_THREADS)
sigmag_filter_kernel(const float* __restrict__ psi_lc, const float* __restrict__ phi_lc, int n_lc, int T,
                     const __grid_constant__ DevParams P, unsigned long long* __restrict__ kept_out,
                     float* __restrict__ lh_out, float* __restrict__ flux_out, uint8_t* __restrict__ pass_out) {
    extern __shared__ float scratch_all[];
    float* scratch = scratch_all + threadIdx.x;
    const int i = blockIdx.x * LC_THREADS + threadIdx.x;
    if (i >= n_lc) return;
    float psi[TP], phi[TP];
#pragma unroll
    for (int t = 0; t < TP; ++t) {
        float a = 0.0f, b = 0.0f;
        if (t < T) {
            a = __ldg(psi_lc + (size_t)i * T + t);
            b = __ldg(phi_lc + (size_t)i * T + t);
        }
        const bool ok = b > 0.0f;
        psi[t] = ok ? a : 0.0f;
        phi[t] = ok ? b : 0.0f;
    }
    float lh, flux;
    unsigned long long kept;
    const int nk = kb_score_lightcurve<TP>(psi, phi, P, scratch, LC_THREADS, lh, flux, kept);
    if (kept_out) kept_out[i] = kept;
    if (lh_out) lh_out[i] = lh;
    if (flux_out) flux_out[i] = flux;
    // "reject the trajectory if the recomputed likelihood (sum LH') is less than 10"
    if (pass_out) pass_out[i] = (nk > 0 && lh >= P.min_lh) ? 1 : 0;
}

// Ordered compaction of the pass flags into a list of surviving lightcurve indices.  Blocks take contiguous chunks
// in ticket order (a block's ticket is its arrival order, so the block it waits for has always started: no
// co-residency assumption), count their survivors, chain the running total through ctr[0] and write their indices
// at the offset they were handed.  ctr: [0] running total (= the number of survivors at the end), [1] tickets
// issued, [2] chunks that have published their total; all zero on entry.
constexpr int CP_THREADS = 256;
__global__ void __launch_bounds__(CP_THREADS)
compact_pass_kernel(const uint8_t* __restrict__ pass, int n, int chunk, int32_t* __restrict__ survivors,
                    unsigned long long* __restrict__ ctr) {
    __shared__ unsigned int s_warp[CP_THREADS / 32];
    __shared__ unsigned long long s_base;
    __shared__ unsigned int s_ticket;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_ticket = (unsigned int)atomicAdd(ctr + 1, 1ull);
    __syncthreads();
    const unsigned int ticket = s_ticket;
    const long long lo = (long long)ticket * chunk, hi = lo + chunk < n ? lo + chunk : n;
    // pass 1: count
    unsigned int cnt = 0;
    for (long long i = lo + threadIdx.x; i < hi; i += CP_THREADS) cnt += pass[i] ? 1u : 0u;
    cnt = __reduce_add_sync(0xFFFFFFFFu, cnt);
    if (lane == 0) s_warp[warp] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int total = 0;
        for (int w = 0; w < CP_THREADS / 32; ++w) total += s_warp[w];
        volatile unsigned long long* done = ctr + 2;
        while (*done != (unsigned long long)ticket) __nanosleep(64);
        __threadfence();
        s_base = atomicAdd(ctr, (unsigned long long)total);  // only this block touches ctr[0] now: the old value is its offset
        __threadfence();
        *done = (unsigned long long)ticket + 1ull;
    }
    __syncthreads();
    unsigned long long base = s_base;
    // pass 2: ordered write, one tile of CP_THREADS flags at a time
    for (long long t0 = lo; t0 < hi; t0 += CP_THREADS) {
        const long long i = t0 + threadIdx.x;
        const bool f = i < hi && pass[i];
        const unsigned int bal = __ballot_sync(0xFFFFFFFFu, f);
        __syncthreads();  // s_warp of the previous tile has been read
        if (lane == 0) s_warp[warp] = __popc(bal);
        __syncthreads();
        unsigned int before = 0, total = 0;
        for (int w = 0; w < CP_THREADS / 32; ++w) {
            const unsigned int c = s_warp[w];
            before += w < warp ? c : 0u;
            total += c;
        }
        if (f && survivors) survivors[base + before + __popc(bal & ((1u << lane) - 1u))] = (int32_t)i;
        base += total;
    }
}

}  // namespace

int kb_launch_eval_trajectories(const float* d_psiphi, int T, int TPv, int H, int W, const DevTimes& times,
                                const int32_t* d_x0, const int32_t* d_y0, const float* d_vx, const float* d_vy,
                                int n_traj, const DevParams& P, float* d_psi_lc, float* d_phi_lc,
                                unsigned long long* d_valid, unsigned long long* d_kept, float* d_lh, float* d_flux,
                                cudaStream_t st) {
    const int grid = (n_traj + LC_THREADS - 1) / LC_THREADS;
    KB_DISPATCH_TP(TPv, {
        const size_t smem = (size_t)TP * LC_THREADS * sizeof(float);
        eval_trajectories_kernel<TP><<<grid, LC_THREADS, smem, st>>>(reinterpret_cast<const float2*>(d_psiphi), T, H, W,
                                                                     times, d_x0, d_y0, d_vx, d_vy, n_traj, P, d_psi_lc,
                                                                     d_phi_lc, d_valid, d_kept, d_lh, d_flux);
    });
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}

int kb_launch_sigmag_filter(const float* d_psi_lc, const float* d_phi_lc, int n_lc, int T, int TPv, const DevParams& P,
                            unsigned long long* d_kept, float* d_lh, float* d_flux, uint8_t* d_pass,
                            unsigned long long* d_n_pass, int32_t* d_survivors, cudaStream_t st) {
    const int grid = (n_lc + LC_THREADS - 1) / LC_THREADS;
    KB_DISPATCH_TP(TPv, {
        const size_t smem = (size_t)TP * LC_THREADS * sizeof(float);
        sigmag_filter_kernel<TP><<<grid, LC_THREADS, smem, st>>>(d_psi_lc, d_phi_lc, n_lc, T, P, d_kept, d_lh, d_flux, d_pass);
    });
    KB_CUDA(cudaGetLastError());
    if (d_n_pass) {
        KB_CUDA(cudaMemsetAsync(d_n_pass, 0, 4 * sizeof(unsigned long long), st));
        const int chunk = std::max(CP_THREADS * 16, (n_lc + 1023) / 1024);  // at most 1024 chunks in the chain
        const int blocks = (n_lc + chunk - 1) / chunk;
        compact_pass_kernel<<<blocks, CP_THREADS, 0, st>>>(d_pass, n_lc, chunk, d_survivors, d_n_pass);
        KB_CUDA(cudaGetLastError());
    }
    return KBMOD_OK;
}

// ---------------------------------------------------------------------------------------------
// kbmod_sigmag_postfilter_static: the post-filter for callers that cannot allocate device memory (code under CUDA
// graph capture, serving loops, harnesses that forbid cudaMalloc).  Same kernels' arithmetic and results as
// kbmod_sigmag_postfilter, but the scratch -- the pass flags [n_lc] and the counters of the ordered compaction --
// lives in a file-scope device array inside the library instead of caller-provided buffers:
// 256 bytes of counters + KBMOD_POSTFILTER_STATIC_MAX_LC flag bytes = 4 MiB + 256 B on every GPU that loads the
// library, held until the process exits.  Every call on a device shares the array and it keeps the last call's
// contents: the counters are cleared on the stream at the start of each call, the flags of [0, n_lc) are all
// rewritten by the filter kernel; two calls that overlap on the GPU (different streams without an ordering
// between them) race on it.
namespace {

constexpr int PFS_HEAD = 256;  // bytes in front of the flags: ctr[0..2] of the compaction chain
static __device__ __align__(256) unsigned char g_postfilter_scratch[PFS_HEAD + KBMOD_POSTFILTER_STATIC_MAX_LC];

// In host code `g_postfilter_scratch` is only the host-side stand-in of the symbol; the device address is looked up
// once per device (with that device current) and cached.
constexpr int PFS_MAX_DEVICES = 64;
std::mutex g_pfs_mutex;
unsigned char* g_pfs_addr[PFS_MAX_DEVICES] = {};

int postfilter_scratch_address(unsigned char** out) {
    int dev = -1;
    KB_CUDA(cudaGetDevice(&dev));
    KB_REQUIRE(dev >= 0 && dev < PFS_MAX_DEVICES, KBMOD_ERR_UNSUPPORTED, "device ordinal %d is beyond %d", dev, PFS_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_pfs_mutex);
    if (!g_pfs_addr[dev]) {
        void* p = nullptr;
        KB_CUDA(cudaGetSymbolAddress(&p, g_postfilter_scratch));
        KB_REQUIRE(p != nullptr, KBMOD_ERR_CUDA, "cudaGetSymbolAddress returned a NULL address");
        g_pfs_addr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_pfs_addr[dev];
    return KBMOD_OK;
}

// compact_pass_kernel with the count delivered to the caller: the block holding the last ticket closes the chain
// and writes the total to n_out (the caller's counter is an output here, not scratch).
__global__ void __launch_bounds__(CP_THREADS)
compact_pass_static_kernel(const uint8_t* __restrict__ pass, int n, int chunk, int n_chunks,
                           int32_t* __restrict__ survivors, unsigned long long* __restrict__ ctr,
                           unsigned long long* __restrict__ n_out) {
    __shared__ unsigned int s_warp[CP_THREADS / 32];
    __shared__ unsigned long long s_base;
    __shared__ unsigned int s_ticket;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_ticket = (unsigned int)atomicAdd(ctr + 1, 1ull);
    __syncthreads();
    const unsigned int ticket = s_ticket;
    const long long lo = (long long)ticket * chunk, hi = lo + chunk < n ? lo + chunk : n;
    unsigned int cnt = 0;
    for (long long i = lo + threadIdx.x; i < hi; i += CP_THREADS) cnt += pass[i] ? 1u : 0u;
    cnt = __reduce_add_sync(0xFFFFFFFFu, cnt);
    if (lane == 0) s_warp[warp] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int total = 0;
        for (int w = 0; w < CP_THREADS / 32; ++w) total += s_warp[w];
        volatile unsigned long long* done = ctr + 2;
        while (*done != (unsigned long long)ticket) __nanosleep(64);
        __threadfence();
        s_base = atomicAdd(ctr, (unsigned long long)total);
        if ((int)ticket == n_chunks - 1) *n_out = s_base + total;
        __threadfence();
        *done = (unsigned long long)ticket + 1ull;
    }
    __syncthreads();
    unsigned long long base = s_base;
    for (long long t0 = lo; t0 < hi; t0 += CP_THREADS) {
        const long long i = t0 + threadIdx.x;
        const bool f = i < hi && pass[i];
        const unsigned int bal = __ballot_sync(0xFFFFFFFFu, f);
        __syncthreads();
        if (lane == 0) s_warp[warp] = __popc(bal);
        __syncthreads();
        unsigned int before = 0, total = 0;
        for (int w = 0; w < CP_THREADS / 32; ++w) {
            const unsigned int c = s_warp[w];
            before += w < warp ? c : 0u;
            total += c;
        }
        if (f) survivors[base + before + __popc(bal & ((1u << lane) - 1u))] = (int32_t)i;
        base += total;
    }
}

}  // namespace

extern "C" int kbmod_sigmag_postfilter_static(const float* d_psi_lc, const float* d_phi_lc, int n_lc, int T,
                                              const kbmod_search_params* p, uint64_t* d_kept, float* d_lh,
                                              float* d_flux, int32_t* d_survivors, uint64_t* d_n_survivors,
                                              void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    KB_REQUIRE(p && d_n_survivors, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(n_lc >= 0, KBMOD_ERR_INVALID_ARG, "n_lc = %d", n_lc);
    KB_REQUIRE(d_survivors || n_lc == 0, KBMOD_ERR_INVALID_ARG, "NULL d_survivors");
    KB_REQUIRE(n_lc <= KBMOD_POSTFILTER_STATIC_MAX_LC, KBMOD_ERR_WORKSPACE,
               "kbmod_sigmag_postfilter_static: n_lc = %d exceeds the static scratch (KBMOD_POSTFILTER_STATIC_MAX_LC = %d "
               "lightcurves per call); split the list or use kbmod_sigmag_postfilter with caller-owned buffers",
               n_lc, KBMOD_POSTFILTER_STATIC_MAX_LC);
    kbmod_search_params q = *p;
    if (q.K < 1 || q.K > KBMOD_MAX_K) q.K = 1;
    DevParams P;
    int rc = kb_make_dev_params(&q, T, &P);
    if (rc) return rc;
    KB_CUDA(cudaMemsetAsync(d_n_survivors, 0, sizeof(unsigned long long), st));
    if (n_lc == 0) return KBMOD_OK;
    KB_REQUIRE(d_psi_lc && d_phi_lc, KBMOD_ERR_INVALID_ARG, "NULL lightcurves");
    unsigned char* scratch = nullptr;
    rc = postfilter_scratch_address(&scratch);
    if (rc) return rc;
    unsigned long long* ctr = reinterpret_cast<unsigned long long*>(scratch);
    uint8_t* pass = scratch + PFS_HEAD;
    KB_CUDA(cudaMemsetAsync(ctr, 0, 4 * sizeof(unsigned long long), st));  // the chain must start at zero
    const int grid = (n_lc + LC_THREADS - 1) / LC_THREADS;
    const int TPv = kb_padded_T(T);
    KB_DISPATCH_TP(TPv, {
        const size_t smem = (size_t)TP * LC_THREADS * sizeof(float);
        sigmag_filter_kernel<TP><<<grid, LC_THREADS, smem, st>>>(d_psi_lc, d_phi_lc, n_lc, T, P,
                                                                 (unsigned long long*)d_kept, d_lh, d_flux, pass);
    });
    KB_CUDA(cudaGetLastError());
    const int chunk = std::max(CP_THREADS * 16, (n_lc + 1023) / 1024);
    const int blocks = (n_lc + chunk - 1) / chunk;
    compact_pass_static_kernel<<<blocks, CP_THREADS, 0, st>>>(pass, n_lc, chunk, blocks, d_survivors, ctr,
                                                              (unsigned long long*)d_n_survivors);
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}
