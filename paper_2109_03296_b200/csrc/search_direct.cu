// (a3)-(a5) direct search: one thread per start pixel walks every velocity, gathers the T samples of the
// trajectory from the padded canvas (one 8-byte (f, m) load per sample, no bounds test; a warp is 32 consecutive x0,
// so each epoch is one 256-byte row segment through L1), runs the sigma-G filter on the register-resident
// lightcurve and keeps its pixel's top-K keys in shared memory.  search_common.cu's finalize_kernel turns the keys
// into the output arrays.
// PAPER.md:L79-L81 (s3), L93-L117 (s3.1), L127-L137 (s3.2); steps 1-4 of kbmod_search in include/kbmod_b200.h.
// This is the evaluator for every trajectory when no threshold prunes (min_lh = -inf) and the implementation the
// pruned kernel must agree with bit for bit.
//
// Instructions per trajectory at T = 26 (round 1: 1600): 7 offset loads + 26 x (IMAD.WIDE + LDG.64 + shift-add of the
// valid bit) gather, 147 x 2 FMNMX sort (half-rate ALU pipe), 26 STS + 3 LDS rank lookup, 26 x (2 FSETP + FFMA + FADD)
// clip-and-sum.  The executed count and the pipe utilisations are in profiles/r2_search_direct_kernel_full.md.
#include <algorithm>

#include "common.cuh"

namespace {

constexpr int SD_BX = 32, SD_BY = 4;  // block = 4 warps, each a 32-pixel row segment
constexpr int SD_THREADS = SD_BX * SD_BY;
#ifndef KB_SD_BLOCKS
#define KB_SD_BLOCKS 5
#endif
// Persistent blocks per SM: a lightcurve is 2 x T registers (f, m), the kernel fits 96 registers and 5 blocks of 128
// threads fill the register file.  The velocity list is walked in an order in which neighbours are neighbours in
// displacement space, so that consecutive velocities of a warp touch overlapping lines.  Measured on configs[2],
// mode (B): 4 / 5 / 6 blocks per SM take 2.33 / 2.29 / 2.32 s (6 blocks: 80 registers, spills); with the 16-byte
// (psi, phi, f, valid) cell of the earlier design (128 registers, 4 blocks) 2.82 s; in list order +0.5 s.
constexpr int SD_BLOCKS_PER_SM = KB_SD_BLOCKS;
// ... for lightcurves of up to 28 epochs.  Longer ones need more registers (2 x T values + the sort's copy; at 96
// registers T = 50 spills 488 bytes per thread): 3 blocks per SM (170 registers).  Measured on configs[3], mode (B),
// T = 50: 5 / 4 / 3 / 2 blocks per SM take 31.5 / 18.8 / 16.4 / 19.1 s.
template <int TP> struct SdCfg {
    static constexpr int blocks = TP <= 28 ? SD_BLOCKS_PER_SM : 3;
};
constexpr int SD_SBW = 8, SD_SBH = 64;  // super-block of tiles: 8 x 32 = 256 pixels wide, 64 x 4 = 256 rows tall

template <int TP>
__global__ void __launch_bounds__(SD_THREADS, SdCfg<TP>::blocks)
search_direct_kernel(const float2* __restrict__ S4, const __grid_constant__ S4Geom G, const int* __restrict__ off,
                     const int* __restrict__ order, int W, int row_begin, int row_end, int n_vel,
                     const __grid_constant__ DevParams P, unsigned long long* __restrict__ keys_out,
                     unsigned long long* __restrict__ next_unit) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* scratch = reinterpret_cast<float*>(smem_raw) + (threadIdx.y * SD_BX + threadIdx.x);  // [TP][threads]
    unsigned long long* list =
        reinterpret_cast<unsigned long long*>(smem_raw + (size_t)TP * SD_THREADS * sizeof(float)) +
        (threadIdx.y * SD_BX + threadIdx.x);  // [K][threads], descending; 0 = empty
    const int K = P.K;
    constexpr int TP4 = (TP + 3) & ~3;
    const int tiles_x = (W + SD_BX - 1) / SD_BX, tiles_y = (row_end - row_begin + SD_BY - 1) / SD_BY;
    // tiles are numbered in compact super-blocks of SD_SBW x SD_SBH tiles (256 x 256 pixels, about one grid's worth), not
    // along whole image rows: the blocks running at one time then cover a square patch, whose displaced copies (blocks
    // drift apart by tens of velocities) still fit L2; in row-major order the same drift spread a 2048-pixel-wide strip
    // over several hundred MB and the kernel read 12.6 TB from DRAM per search.
    const int sb_per_row = (tiles_x + SD_SBW - 1) / SD_SBW;
    const int n_sb = sb_per_row * ((tiles_y + SD_SBH - 1) / SD_SBH);
    // Work units are the 32-pixel row segments of the tiles, handed out to the warps from a global counter in tile
    // order (the warps in flight at one time work on neighbouring rows of neighbouring tiles): trajectories near the
    // edges the velocities point away from leave the image early and cost a fraction of an interior row, so a static
    // split leaves a fifth of the warp slots idle towards the end (measured on configs[2], mode (B): 2.23 s static,
    // 2.22 s with twice as many blocks in two waves, 1.78 s this way).
    const unsigned int n_units = (unsigned int)(n_sb * SD_SBW * SD_SBH) * SD_BY;
    for (;;) {
        unsigned int u = 0;
        if (threadIdx.x == 0) u = (unsigned int)atomicAdd(next_unit, 1ull);
        u = __shfl_sync(0xFFFFFFFFu, u, 0);
        if (u >= n_units) break;
        const int slot = (int)(u / SD_BY), r = (int)(u % SD_BY);
        const int sb = slot / (SD_SBW * SD_SBH), in = slot - sb * (SD_SBW * SD_SBH);
        const int sby = sb / sb_per_row, sbx = sb - sby * sb_per_row;
        const int ty = sby * SD_SBH + in / SD_SBW, tx = sbx * SD_SBW + in % SD_SBW;
        if (tx >= tiles_x || ty >= tiles_y) continue;  // warp-uniform
        const int x0 = tx * SD_BX + threadIdx.x;
        const int y0 = row_begin + ty * SD_BY + r;
        if (y0 >= row_end) continue;  // warp-uniform: the last tile row of the band may be partial
        const bool active = x0 < W;
        // lanes past the edge evaluate the edge pixel again and write nothing: the warp stays whole
        const int xc = min(x0, W - 1), yc = y0;
        for (int k = 0; k < K; ++k) list[k * SD_THREADS] = 0ull;
        unsigned long long kth = 0ull;  // key of slot K-1: only a larger key enters the list
        const unsigned int base = (unsigned int)(yc + G.pyn) * (unsigned int)G.Wp + (unsigned int)(xc + G.pxn);
#pragma unroll 1
        for (int i = 0; i < n_vel; ++i) {
            __syncwarp();  // re-converge after the divergent top-K insertion of the previous velocity
            const int v = __ldg(order + i);
            float f[TP], m[TP], sp, sf;
            int n;
            kb_gather_s4<TP>(S4, base, reinterpret_cast<const int4*>(off + (size_t)v * TP4), f, m, n);  // uniform row
            const int nk = kb_score_s4<TP, false>(f, m, n, P, scratch, SD_THREADS, sp, sf);
            if (nk == 0) continue;
            const float lh = kb_lh_of(sp, sf);
            if (!(lh >= P.min_lh)) continue;
            const unsigned long long key = kb_topk_key(lh, v);
            if (key <= kth) continue;
            // insert: the list is sorted by key, i.e. by (L' desc, vel_idx asc), whatever the order of arrival
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
        __syncwarp();
        if (active) {
            unsigned long long* out = keys_out + ((size_t)(y0 - row_begin) * W + x0) * K;
            for (int k = 0; k < K; ++k) out[k] = list[k * SD_THREADS];
        }
    }
}

}  // namespace

int kb_launch_search_direct(int TPv, const void* d_S4, const S4Geom& G, const int* d_off, const int* d_order, int W,
                            int row_begin, int row_end, int n_vel, const DevParams& P, unsigned long long* d_keys,
                            unsigned long long* d_next_unit, cudaStream_t st) {
    const int n_rows = row_end - row_begin;
    if (n_rows <= 0) return KBMOD_OK;
    int n_sm = 148, dev = 0;
    KB_CUDA(cudaGetDevice(&dev));
    KB_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    const dim3 block(SD_BX, SD_BY);
    const int n_tiles = ((W + SD_BX - 1) / SD_BX) * ((n_rows + SD_BY - 1) / SD_BY);
    KB_CUDA(cudaMemsetAsync(d_next_unit, 0, sizeof(unsigned long long), st));
    KB_DISPATCH_TP(TPv, {
        const dim3 grid(std::min(n_tiles, n_sm * SdCfg<TP>::blocks));
        const size_t smem = (size_t)TP * SD_THREADS * sizeof(float) + (size_t)P.K * SD_THREADS * sizeof(unsigned long long);
        KB_CUDA(cudaFuncSetAttribute(search_direct_kernel<TP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        search_direct_kernel<TP><<<grid, block, smem, st>>>(reinterpret_cast<const float2*>(d_S4), G, d_off, d_order, W,
                                                            row_begin, row_end, n_vel, P, d_keys, d_next_unit);
    });
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}
