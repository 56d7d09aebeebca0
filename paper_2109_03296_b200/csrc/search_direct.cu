// (a3)-(a5) direct search: one thread per start pixel walks every velocity, gathers the T samples of the
// trajectory from the padded S4 canvas (one 16-byte load per sample, no bounds test; a warp is 32 consecutive x0,
// so each epoch is one 512-byte row segment through L1), runs the sigma-G filter on the register-resident
// lightcurve and keeps its pixel's top-K keys in shared memory.  search_common.cu's finalize_kernel turns the keys
// into the output arrays.
// PAPER.md:L79-L81 (s3), L93-L117 (s3.1), L127-L137 (s3.2); steps 1-4 of kbmod_search in include/kbmod_b200.h.
// This is the evaluator for every trajectory when no threshold prunes (min_lh = -inf) and the implementation the
// pruned kernel must agree with bit for bit.
//
// Instruction budget per trajectory at T = 26 (the binding resource is instruction issue; the half-rate ALU pipe
// takes the 147 FMNMX of the network and the 52 FSETP of the clip): 7 offset loads + 26 x (IMAD.WIDE + LDG.128 +
// IADD) gather, 147 x (FMNMX + IADD3) sort, 26 STS + 3 LDS rank lookup, 26 x 5 clip-and-sum.
#include "common.cuh"

namespace {

constexpr int SD_BX = 32, SD_BY = 4;  // block = 4 warps, each a 32-pixel row segment
constexpr int SD_THREADS = SD_BX * SD_BY;

template <int TP>
__global__ void __launch_bounds__(SD_THREADS)
search_direct_kernel(const float4* __restrict__ S4, const __grid_constant__ S4Geom G, const int* __restrict__ off,
                     int W, int row_begin, int row_end, int n_vel, const __grid_constant__ DevParams P,
                     unsigned long long* __restrict__ keys_out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* scratch = reinterpret_cast<float*>(smem_raw) + (threadIdx.y * SD_BX + threadIdx.x);  // [TP][threads]
    unsigned long long* list =
        reinterpret_cast<unsigned long long*>(smem_raw + (size_t)TP * SD_THREADS * sizeof(float)) +
        (threadIdx.y * SD_BX + threadIdx.x);  // [K][threads], descending; 0 = empty

    const int x0 = blockIdx.x * SD_BX + threadIdx.x;
    const int y0 = row_begin + blockIdx.y * SD_BY + threadIdx.y;
    if (x0 >= W || y0 >= row_end) return;
    const int K = P.K;
    for (int k = 0; k < K; ++k) list[k * SD_THREADS] = 0ull;
    unsigned long long kth = 0ull;  // key of slot K-1: only a larger key enters the list
    const unsigned int base = (unsigned int)(y0 + G.pyn) * (unsigned int)G.Wp + (unsigned int)(x0 + G.pxn);
    constexpr int TP4 = (TP + 3) & ~3;

    const unsigned warp_mask = __activemask();  // lanes past the right edge have left
#pragma unroll 1
    for (int v = 0; v < n_vel; ++v) {
        __syncwarp(warp_mask);  // re-converge after the divergent top-K insertion of the previous velocity
        float psi[TP], phi[TP], f[TP], sp, sf;
        int n;
        kb_gather_s4<TP>(S4, base, reinterpret_cast<const int4*>(off + (size_t)v * TP4), psi, phi, f, n);  // uniform row
        const int nk = kb_score_s4<TP>(psi, phi, f, n, P, scratch, SD_THREADS, sp, sf);
        if (nk == 0) continue;
        const float lh = kb_lh_of(sp, sf);
        if (!(lh >= P.min_lh)) continue;
        const unsigned long long key = kb_topk_key(lh, v);
        if (key <= kth) continue;
        // insert: the list is sorted by key, i.e. by (L' desc, vel_idx asc)
        int pos = K - 1;
        while (pos > 0) {
            const unsigned long long up = list[(pos - 1) * SD_THREADS];
            if (up >= key) break;
            list[pos * SD_THREADS] = up;
            --pos;
        }
        list[pos * SD_THREADS] = key;
        kth = list[(K - 1) * SD_THREADS];
    }
    unsigned long long* out = keys_out + ((size_t)(y0 - row_begin) * W + x0) * K;
    for (int k = 0; k < K; ++k) out[k] = list[k * SD_THREADS];
}

}  // namespace

int kb_launch_search_direct(int TPv, const void* d_S4, const S4Geom& G, const int* d_off, int W, int row_begin,
                            int row_end, int n_vel, const DevParams& P, unsigned long long* d_keys, cudaStream_t st) {
    const int n_rows = row_end - row_begin;
    if (n_rows <= 0) return KBMOD_OK;
    const dim3 block(SD_BX, SD_BY);
    const dim3 grid((W + SD_BX - 1) / SD_BX, (n_rows + SD_BY - 1) / SD_BY);
    KB_DISPATCH_TP(TPv, {
        const size_t smem = (size_t)TP * SD_THREADS * sizeof(float) + (size_t)P.K * SD_THREADS * sizeof(unsigned long long);
        KB_CUDA(cudaFuncSetAttribute(search_direct_kernel<TP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        search_direct_kernel<TP><<<grid, block, smem, st>>>(reinterpret_cast<const float4*>(d_S4), G, d_off, W, row_begin,
                                                            row_end, n_vel, P, d_keys);
    });
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}
