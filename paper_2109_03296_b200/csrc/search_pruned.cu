// (a3)-(a5) pruned search.  Same results as search_direct.cu; the full sigma-G evaluation runs only
// for trajectories whose EXACT upper bound reaches the threshold min_lh (trajectories
// with a recomputed likelihood below 10 are rejected; L115: only sum-LH > 10 leave the GPU).
//
// Bound.  For any kept set S produced by the sigma-G filter,
//     L' = sum_S psi / sqrt(sum_S phi)  <=  sum_valid max(psi,0) / sqrt(m(n) * min_valid phi)  =: U
// because sum_S psi <= sum_valid psi_+, and S always contains every epoch whose value lies between
// the two percentiles (the clip window is the median +- n_sigma*C*(P_hi-P_lo) with n_sigma*C >= 1 and
// P_lo <= P_50 <= P_hi), so |S| >= m(n) = rank_hi(n) - rank_lo(n) + 1 and sum_S phi >= m(n) min phi.
// U needs one float2 per trajectory-epoch: (a, q) = (psi_+, -1/sqrt(phi)), zero where invalid:
//     A += a;  qmin = min(qmin, q);  n += (q < 0)        U = A * (-qmin) / sqrt(m(n))
//
// Phase 1 (where the time goes): epoch-outer; a CTA owns a 64x16 tile of start pixels and a group
// of 16 neighbouring velocities; for each epoch the tile (+) the group's displacement bounding box
// is staged by TMA (zero fill outside the image = the off-chip rule) into a double-buffered shared
// memory region and every thread gathers its 2 pixels x 16 velocities from it (8 B per
// trajectory-epoch evaluation, conflict-free LDS.64).  Phase 2: (pixel, velocity) pairs whose bound
// reaches min_lh are compacted into a shared-memory queue and evaluated exactly by the same device
// function as the direct kernel, gathering from the psi/phi stack in L2.  Results enter the per-pixel
// top-K through a cascade of 64-bit atomicMax on (orderable L', ~vel_idx) keys; a last kernel turns
// keys into the four output arrays.
#include <algorithm>
#include <vector>

#include "common.cuh"
#include "tma.cuh"

namespace {

constexpr int PR_TW = 64, PR_TH = 16;      // tile of start pixels per CTA
constexpr int PR_G = 16;                   // velocities per group
constexpr int PR_THREADS = 512;            // 16 warps; thread = (x, y) and (x+32, y)
constexpr int PR_RB = 8;                   // rows per TMA box
constexpr int PR_NPITCH = 12;              // tensor maps: pitch = 64 + 16*k elements, k < 12  (<= 240)
constexpr int PR_BUF_BYTES = 96 * 1024;    // one staging buffer
constexpr int PR_MAXT = KBMOD_MAX_T;

struct __align__(8) GroupEpoch {
    int16_t ox, oy;    // region origin relative to the tile origin (min dx, min dy of the group)
    uint16_t pitch_k;  // tensor map / pitch index
    uint16_t n_box;    // boxes of PR_RB rows; 0xFFFF in epoch 0 marks a group that cannot be staged
};

struct PrunedTables {  // device pointers into the workspace
    const int32_t* gvel;     // [n_groups][PR_G]  velocity index or -1
    const GroupEpoch* ge;    // [n_groups][T]
    const int32_t* offs;     // [n_groups][T][PR_G] element offset inside the staged region
    int n_groups;
};

struct TensorMaps {
    CUtensorMap m[PR_NPITCH];
};

struct BoundParams {
    float minv[KBMOD_MAX_T + 1];  // (1 + eps) / sqrt(m(n))
};

// ---------------------------------------------------------------------------------------------
// bound planes: B[t][y][x] = (psi_+, -(1+eps)/sqrt(phi)) for valid pixels, (0, 0) otherwise; row pitch Wp
__global__ void bound_plane_kernel(const float2* __restrict__ psiphi, float2* __restrict__ B, int W, int Wp,
                                   size_t rows /* T*H */) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows * (size_t)Wp) return;
    const size_t r = i / Wp;
    const int x = (int)(i - r * Wp);
    float2 o = make_float2(0.0f, 0.0f);
    if (x < W) {
        const float2 s = __ldg(psiphi + r * W + x);
        if (s.y > 0.0f) {
            // 1/sqrt(phi) rounded up: rsqrtf is within 2 ulp, the factor 1 + 2^-20 covers it
            o.x = fmaxf(s.x, 0.0f);
            o.y = -(rsqrtf(s.y) * 1.00000095367431640625f);
        }
    }
    B[i] = o;
}

__device__ __forceinline__ unsigned int orderable(float f) {
    const unsigned int u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float unorderable(unsigned int u) {
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7FFFFFFFu) : ~u);
}

// insert into a descending list of K keys shared by all CTAs (empty = 0): each slot ends up
// holding the maximum of everything that reached it, so the list is the top-K of all insertions.
__device__ __forceinline__ void topk_insert(unsigned long long* keys, int K, unsigned long long key) {
    for (int k = 0; k < K && key != 0ull; ++k) {
        const unsigned long long old = atomicMax(keys + k, key);
        key = old < key ? old : key;  // whichever lost moves on to the next slot
    }
}

// ---------------------------------------------------------------------------------------------
// shared memory carve-up (dynamic): two staging buffers, then the per-item tables
struct PrSmemTail {
    int32_t offs[PR_MAXT][PR_G];
    GroupEpoch ge[PR_MAXT];
    int32_t gvel[PR_G];
    uint64_t full[2];
    unsigned int qcount;
};
constexpr size_t PR_SMEM_BYTES = 2 * (size_t)PR_BUF_BYTES + sizeof(PrSmemTail);

template <int TP>
__global__ void __launch_bounds__(PR_THREADS, 1)
search_pruned_kernel(const __grid_constant__ TensorMaps maps, const float2* __restrict__ psiphi, int T, int H, int W,
                     const DispEntry* __restrict__ tab, const __grid_constant__ PrunedTables tb,
                     const __grid_constant__ DevParams P, const __grid_constant__ BoundParams BP,
                     unsigned long long* __restrict__ keys, unsigned long long* __restrict__ stats) {
    extern __shared__ __align__(1024) unsigned char smem[];
    float2* buf0 = reinterpret_cast<float2*>(smem);
    float2* buf1 = reinterpret_cast<float2*>(smem + PR_BUF_BYTES);
    PrSmemTail& S = *reinterpret_cast<PrSmemTail*>(smem + 2 * (size_t)PR_BUF_BYTES);
    unsigned short* queue = reinterpret_cast<unsigned short*>(smem);         // phase 2: aliases buf0
    float* scratch_all = reinterpret_cast<float*>(smem + PR_BUF_BYTES);      // phase 2: aliases buf1
    constexpr int P2_THREADS = (TP <= 48) ? PR_THREADS : PR_THREADS / 2;     // scratch is [TP][P2_THREADS] floats

    const int tid = threadIdx.x;
    const int tx = tid & 31, ty = tid >> 5;
    if (tid == 0) {
        kb_mbar_init(&S.full[0], 1);
        kb_mbar_init(&S.full[1], 1);
        kb_fence_barrier_init();
        for (int k = 0; k < PR_NPITCH; ++k) kb_prefetch_tensormap(&maps.m[k]);
    }
    __syncthreads();

    const int tiles_x = (W + PR_TW - 1) / PR_TW, tiles_y = (H + PR_TH - 1) / PR_TH;
    const int n_tiles = tiles_x * tiles_y;
    // tiles are taken in compact blocks of gridDim.x tiles (4 tile columns wide) so that the CTAs
    // running at the same time share their staged regions in L2
    const int need = P.min_obs > 1 ? P.min_obs : 1;
    unsigned int it = 0;  // epochs staged so far by this CTA: buffer = it & 1, parity = (it >> 1) & 1
    unsigned long long n_eval = 0;

    for (int tile_lin = blockIdx.x; tile_lin < n_tiles; tile_lin += gridDim.x) {
        // column-block order: 4 tile columns x all tile rows, then the next 4 columns
        const int cb = tile_lin / (4 * tiles_y), rem = tile_lin - cb * 4 * tiles_y;
        const int cols_here = min(4, tiles_x - cb * 4);
        const int tyi = rem / cols_here, txi = cb * 4 + rem - tyi * cols_here;
        const int tile_x0 = txi * PR_TW, tile_y0 = tyi * PR_TH;
        const int px0 = tile_x0 + tx, py0 = tile_y0 + ty;  // this thread's pixels: (px0, py0), (px0+32, py0)

        for (int g = 0; g < tb.n_groups; ++g) {
            __syncthreads();  // previous item completely done (tables, queue, scratch)
            for (int i = tid; i < T * PR_G; i += PR_THREADS) S.offs[i / PR_G][i % PR_G] = tb.offs[(size_t)g * T * PR_G + i];
            if (tid < T) S.ge[tid] = tb.ge[(size_t)g * T + tid];
            if (tid < PR_G) S.gvel[tid] = tb.gvel[(size_t)g * PR_G + tid];
            if (tid == 0) S.qcount = 0;
            kb_fence_proxy_async();  // phase-2 st.shared into the buffers happen-before the next TMA writes
            __syncthreads();
            const bool stageable = S.ge[0].n_box != 0xFFFFu;

            if (stageable) {
                float A[2][PR_G], Q[2][PR_G];
                int N[2][PR_G];
#pragma unroll
                for (int j = 0; j < PR_G; ++j) {
                    A[0][j] = A[1][j] = 0.0f;
                    Q[0][j] = Q[1][j] = 0.0f;
                    N[0][j] = N[1][j] = 0;
                }
                auto issue = [&](int t, unsigned int slot) {
                    const GroupEpoch e = S.ge[t];
                    const int pitch = PR_TW + 16 * e.pitch_k;
                    const unsigned int box_bytes = (unsigned int)pitch * PR_RB * sizeof(float2);
                    unsigned char* dst = smem + (size_t)slot * PR_BUF_BYTES;
                    kb_mbar_expect_tx(&S.full[slot], box_bytes * e.n_box);
                    for (int b = 0; b < e.n_box; ++b)
                        kb_tma_load_3d(dst + (size_t)b * box_bytes, &maps.m[e.pitch_k], tile_x0 + e.ox,
                                       tile_y0 + e.oy + b * PR_RB, t, &S.full[slot]);
                };
                if (tid == 0) issue(0, it & 1);
#pragma unroll 1
                for (int t = 0; t < T; ++t) {
                    __syncthreads();  // everyone finished reading buffer (it+1)&1 (epoch t-1)
                    if (tid == 0 && t + 1 < T) issue(t + 1, (it + 1) & 1);
                    kb_mbar_wait(&S.full[it & 1], (it >> 1) & 1);
                    const float2* buf = (it & 1) ? buf1 : buf0;
                    const int pitch = PR_TW + 16 * S.ge[t].pitch_k;
                    const float2* base = buf + ty * pitch + tx;
#pragma unroll
                    for (int j = 0; j < PR_G; ++j) {
                        const float2* p = base + S.offs[t][j];
                        const float2 v0 = p[0], v1 = p[32];
                        A[0][j] += v0.x;
                        Q[0][j] = fminf(Q[0][j], v0.y);
                        N[0][j] += (int)(__float_as_uint(v0.y) >> 31);
                        A[1][j] += v1.x;
                        Q[1][j] = fminf(Q[1][j], v1.y);
                        N[1][j] += (int)(__float_as_uint(v1.y) >> 31);
                    }
                    ++it;
                }
                __syncthreads();  // all reads of the staging buffers done: the queue may overwrite buf0
                // bound test; survivors -> queue entry = (pixel-in-tile << 4) | velocity-in-group
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const bool in_img = (px0 + 32 * h) < W && py0 < H;
#pragma unroll
                    for (int j = 0; j < PR_G; ++j) {
                        const int n = N[h][j];
                        const float U = A[h][j] * (-Q[h][j]) * BP.minv[n];
                        if (in_img && n >= need && U >= P.min_lh && S.gvel[j] >= 0) {
                            const unsigned int pos = atomicAdd(&S.qcount, 1u);
                            queue[pos] = (unsigned short)(((ty * PR_TW + tx + 32 * h) << 4) | j);
                        }
                    }
                }
            } else {
                // group cannot be staged (its displacement box does not fit): every pair is evaluated
                for (int i = tid; i < PR_TW * PR_TH * PR_G; i += PR_THREADS) {
                    const int pix = i >> 4, j = i & 15;
                    const bool in_img = (tile_x0 + (pix & (PR_TW - 1))) < W && (tile_y0 + pix / PR_TW) < H;
                    if (in_img && S.gvel[j] >= 0) queue[atomicAdd(&S.qcount, 1u)] = (unsigned short)i;
                }
            }
            __syncthreads();
            // ---- phase 2: exact evaluation of the queued pairs (the direct kernel's device function)
            const unsigned int qn = S.qcount;
            if (tid == 0) n_eval += qn;
            for (unsigned int q0 = 0; q0 < qn; q0 += P2_THREADS) {
                const unsigned int qi = q0 + tid;
                if (tid < P2_THREADS && qi < qn) {
                    const unsigned int e = queue[qi];
                    const int pix = e >> 4, j = e & 15;
                    const int x0 = tile_x0 + (pix & (PR_TW - 1)), y0 = tile_y0 + pix / PR_TW;
                    const int v = S.gvel[j];
                    const DispEntry* row = tab + (size_t)v * TP;
                    const int pixlin = y0 * W + x0;
                    float psi[TP], phi[TP];
#pragma unroll
                    for (int t = 0; t < TP; ++t) {
                        const DispEntry d = row[t];
                        const int x = x0 + d.dx, y = y0 + d.dy;
                        float2 s = make_float2(0.0f, 0.0f);
                        if ((unsigned)x < (unsigned)W && (unsigned)y < (unsigned)H) s = __ldg(psiphi + (pixlin + d.off));
                        const bool ok = s.y > 0.0f;
                        psi[t] = ok ? s.x : 0.0f;
                        phi[t] = ok ? s.y : 0.0f;
                    }
                    float lh, flux;
                    unsigned long long kept;
                    const int nk = kb_score_lightcurve<TP>(psi, phi, P, scratch_all + tid, P2_THREADS, lh, flux, kept);
                    if (nk > 0 && lh >= P.min_lh) {
                        const unsigned long long key =
                            ((unsigned long long)orderable(lh) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned)v);
                        topk_insert(keys + (size_t)pixlin * P.K, P.K, key);
                    }
                }
            }
        }
    }
    if (tid == 0 && n_eval) atomicAdd(stats, n_eval);
}

// ---------------------------------------------------------------------------------------------
// keys -> output arrays.  One thread per (pixel, slot); a filled slot is re-evaluated to get flux
// and n_obs (the key carries L' and the velocity index only).
constexpr int FIN_THREADS = 128;

template <int TP>
__global__ void __launch_bounds__(FIN_THREADS)
finalize_kernel(const unsigned long long* __restrict__ keys, const float2* __restrict__ psiphi, int H, int W,
                const DispEntry* __restrict__ tab, const __grid_constant__ DevParams P, float* __restrict__ out_lh,
                float* __restrict__ out_flux, int32_t* __restrict__ out_vel, int32_t* __restrict__ out_nobs) {
    extern __shared__ float scratch_all[];
    const size_t i = (size_t)blockIdx.x * FIN_THREADS + threadIdx.x;
    const size_t total = (size_t)H * W * P.K;
    if (i >= total) return;
    const unsigned long long key = keys[i];
    float lh = -CUDART_INF_F, flux = 0.0f;
    int vel = -1, nobs = 0;
    if (key != 0ull) {
        vel = (int)(0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull));
        const int pixlin = (int)(i / P.K);
        const int y0 = pixlin / W, x0 = pixlin - y0 * W;
        const DispEntry* row = tab + (size_t)vel * TP;
        float psi[TP], phi[TP];
#pragma unroll
        for (int t = 0; t < TP; ++t) {
            const DispEntry d = row[t];
            const int x = x0 + d.dx, y = y0 + d.dy;
            float2 s = make_float2(0.0f, 0.0f);
            if ((unsigned)x < (unsigned)W && (unsigned)y < (unsigned)H) s = __ldg(psiphi + (pixlin + d.off));
            const bool ok = s.y > 0.0f;
            psi[t] = ok ? s.x : 0.0f;
            phi[t] = ok ? s.y : 0.0f;
        }
        unsigned long long kept;
        nobs = kb_score_lightcurve<TP>(psi, phi, P, scratch_all + threadIdx.x, FIN_THREADS, lh, flux, kept);
    }
    out_lh[i] = lh;
    out_flux[i] = flux;
    out_vel[i] = vel;
    out_nobs[i] = nobs;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
kb_encode_tiled_fn kb_get_encode_tiled() {
    static kb_encode_tiled_fn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (kb_encode_tiled_fn)p;
    }
    return fn;
}

// ---------------------------------------------------------------------------------------------
// host planner: velocity grouping (k-d bisection of the displacement at the epoch farthest from
// times[0]) and the per-(group, epoch) staging geometry
namespace {

void kd_groups(std::vector<int>& idx, int lo, int hi, const std::vector<int>& px, const std::vector<int>& py,
               std::vector<std::pair<int, int>>& leaves) {
    const int n = hi - lo;
    if (n <= PR_G) {
        leaves.push_back({lo, hi});
        return;
    }
    int x0 = INT32_MAX, x1 = INT32_MIN, y0 = INT32_MAX, y1 = INT32_MIN;
    for (int i = lo; i < hi; ++i) {
        x0 = std::min(x0, px[idx[i]]); x1 = std::max(x1, px[idx[i]]);
        y0 = std::min(y0, py[idx[i]]); y1 = std::max(y1, py[idx[i]]);
    }
    const bool by_x = (x1 - x0) >= (y1 - y0);
    std::stable_sort(idx.begin() + lo, idx.begin() + hi, [&](int a, int b) {
        return by_x ? (px[a] != px[b] ? px[a] < px[b] : py[a] < py[b]) : (py[a] != py[b] ? py[a] < py[b] : px[a] < px[b]);
    });
    const int ng = (n + PR_G - 1) / PR_G;
    const int half = (ng / 2) * PR_G;  // split at a multiple of the group size: all leaves but one are full
    kd_groups(idx, lo, lo + half, px, py, leaves);
    kd_groups(idx, lo + half, hi, px, py, leaves);
}

}  // namespace

size_t kb_pruned_workspace_bytes(int T, int H, int W, int n_vel, int K) {
    const size_t ng = ((size_t)n_vel + PR_G - 1) / PR_G;
    const size_t Wp = ((size_t)W + 1) & ~(size_t)1;
    auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
    return al(ng * PR_G * 4) + al(ng * T * sizeof(GroupEpoch)) + al(ng * T * PR_G * 4) + al((size_t)T * H * Wp * 8) +
           al((size_t)H * W * K * 8);
}

// m(n): a lower bound on the number of epochs the sigma-G filter keeps out of n valid ones; 0 = no bound
static bool bound_min_kept(const kbmod_search_params* p, const DevParams& P, int T, BoundParams* bp) {
    const float prod = p->n_sigma * p->sigmag_coeff;
    for (int n = 0; n <= KBMOD_MAX_T; ++n) {
        int m = 1;
        if (n >= 1 && n <= T) {
            if (!P.sigmag_enable) m = n;
            else if (prod >= 1.001f && p->pct_lo <= 50.0f && p->pct_hi >= 50.0f) m = P.rk_hi[n] - P.rk_lo[n] + 1;
            else if (prod >= 0.0f && p->n_sigma >= 0.0f) m = 1;
            else return false;
        }
        bp->minv[n] = (float)(1.00003 / sqrt((double)m));  // + slack for the float32 sum and product
    }
    return true;
}

int kb_launch_search_pruned(const float* d_psiphi, int T, int TPv, int H, int W, const DispEntry* d_tab,
                            const int32_t* h_dx, const int32_t* h_dy, int n_vel, const kbmod_search_params* p,
                            const DevParams& P, float* d_lh, float* d_flux, int32_t* d_vel, int32_t* d_nobs,
                            void* d_ws, size_t ws_bytes, unsigned long long* d_stats, cudaStream_t st, int plan_only,
                            double* plan_stats, int* n_launches) {
    BoundParams bp;
    if (!bound_min_kept(p, P, T, &bp)) {
        kb_set_error("pruned search needs n_sigma >= 0 and n_sigma*coeff >= 0");
        return KBMOD_ERR_UNSUPPORTED;
    }
    const int ng = (n_vel + PR_G - 1) / PR_G;
    // ---- grouping
    int t_far = 0;
    {   // epoch with the largest displacement spread
        long long best = -1;
        for (int t = 0; t < T; ++t) {
            long long s = 0;
            for (int v = 0; v < n_vel; v += std::max(1, n_vel / 64)) s += llabs((long long)h_dx[(size_t)v * T + t]) + llabs((long long)h_dy[(size_t)v * T + t]);
            if (s > best) { best = s; t_far = t; }
        }
    }
    std::vector<int> idx(n_vel), px(n_vel), py(n_vel);
    for (int v = 0; v < n_vel; ++v) {
        idx[v] = v;
        px[v] = std::max(-40000, std::min(40000, h_dx[(size_t)v * T + t_far]));
        py[v] = std::max(-40000, std::min(40000, h_dy[(size_t)v * T + t_far]));
    }
    std::vector<std::pair<int, int>> leaves;
    if (n_vel > 0) kd_groups(idx, 0, n_vel, px, py, leaves);
    std::vector<int32_t> gvel((size_t)ng * PR_G, -1), offs((size_t)ng * T * PR_G, 0);
    std::vector<GroupEpoch> ge((size_t)ng * T);
    double staged = 0.0, evals = 0.0;
    int n_unstageable = 0;
    for (int g = 0; g < ng; ++g) {
        const int lo = leaves[g].first, cnt = leaves[g].second - leaves[g].first;
        for (int j = 0; j < cnt; ++j) gvel[(size_t)g * PR_G + j] = idx[lo + j];
        bool ok = true;
        double g_staged = 0.0;
        for (int t = 0; t < T && ok; ++t) {
            int x0 = INT32_MAX, x1 = INT32_MIN, y0 = INT32_MAX, y1 = INT32_MIN;
            for (int j = 0; j < cnt; ++j) {
                const int v = idx[lo + j];
                const int dx = h_dx[(size_t)v * T + t], dy = h_dy[(size_t)v * T + t];
                x0 = std::min(x0, dx); x1 = std::max(x1, dx); y0 = std::min(y0, dy); y1 = std::max(y1, dy);
            }
            // TMA: the box must start on a 16-byte boundary, i.e. at an even x for 8-byte elements (an odd
            // start raises an illegal-instruction fault on sm_100a); tile origins are multiples of 64
            x0 -= (x0 & 1);
            const long long bw = (long long)x1 - x0 + PR_TW, bh = (long long)y1 - y0 + PR_TH;
            const long long pk = (bw - PR_TW + 15) / 16, nb = (bh + PR_RB - 1) / PR_RB;
            const long long bytes = (PR_TW + 16 * pk) * PR_RB * nb * 8;
            if (pk >= PR_NPITCH || bytes > PR_BUF_BYTES || x0 < -30000 || x1 > 30000 || y0 < -30000 || y1 > 30000) {
                ok = false;
                break;
            }
            GroupEpoch e;
            e.ox = (int16_t)x0; e.oy = (int16_t)y0; e.pitch_k = (uint16_t)pk; e.n_box = (uint16_t)nb;
            ge[(size_t)g * T + t] = e;
            const int pitch = PR_TW + 16 * (int)pk;
            for (int j = 0; j < cnt; ++j) {
                const int v = idx[lo + j];
                offs[((size_t)g * T + t) * PR_G + j] = (h_dy[(size_t)v * T + t] - y0) * pitch + (h_dx[(size_t)v * T + t] - x0);
            }
            g_staged += (double)bytes;
        }
        if (!ok) {
            for (int t = 0; t < T; ++t) ge[(size_t)g * T + t] = GroupEpoch{0, 0, 0, 0xFFFF};
            ++n_unstageable;
        } else {
            staged += g_staged;
            evals += (double)PR_TW * PR_TH * cnt * T;
        }
    }
    if (plan_stats) {
        plan_stats[0] = ng ? (double)n_unstageable / ng : 0.0;  // fraction of groups that cannot be staged
        plan_stats[1] = evals > 0 ? staged / evals : 0.0;       // staged bytes per evaluation
    }
    if (plan_only) return KBMOD_OK;

    // ---- workspace carve-up
    auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
    const size_t Wp = ((size_t)W + 1) & ~(size_t)1;
    char* w = (char*)d_ws;
    size_t o = 0;
    int32_t* d_gvel = (int32_t*)(w + o);        o += al((size_t)ng * PR_G * 4);
    GroupEpoch* d_ge = (GroupEpoch*)(w + o);    o += al((size_t)ng * T * sizeof(GroupEpoch));
    int32_t* d_offs = (int32_t*)(w + o);        o += al((size_t)ng * T * PR_G * 4);
    float2* d_B = (float2*)(w + o);             o += al((size_t)T * H * Wp * 8);
    unsigned long long* d_keys = (unsigned long long*)(w + o);
    o += al((size_t)H * W * P.K * 8);
    KB_REQUIRE(o <= ws_bytes, KBMOD_ERR_WORKSPACE, "pruned search workspace: need %zu, have %zu", o, ws_bytes);
    KB_REQUIRE((double)T * H * Wp < 2147483648.0, KBMOD_ERR_UNSUPPORTED, "T*H*Wp exceeds 2^31");

    if (ng > 0) {
        KB_CUDA(cudaMemcpyAsync(d_gvel, gvel.data(), gvel.size() * 4, cudaMemcpyHostToDevice, st));
        KB_CUDA(cudaMemcpyAsync(d_ge, ge.data(), ge.size() * sizeof(GroupEpoch), cudaMemcpyHostToDevice, st));
        KB_CUDA(cudaMemcpyAsync(d_offs, offs.data(), offs.size() * 4, cudaMemcpyHostToDevice, st));
    }
    KB_CUDA(cudaMemsetAsync(d_keys, 0, (size_t)H * W * P.K * 8, st));

    // ---- tensor maps over the bound planes: uint64 elements, dims {Wp, H, T}
    kb_encode_tiled_fn enc = kb_get_encode_tiled();
    KB_REQUIRE(enc != nullptr, KBMOD_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
    TensorMaps maps;
    for (int k = 0; k < PR_NPITCH; ++k) {
        cuuint64_t dims[3] = {(cuuint64_t)Wp, (cuuint64_t)H, (cuuint64_t)T};
        cuuint64_t strides[2] = {(cuuint64_t)Wp * 8, (cuuint64_t)Wp * 8 * (cuuint64_t)H};
        cuuint32_t box[3] = {(cuuint32_t)(PR_TW + 16 * k), (cuuint32_t)PR_RB, 1};
        cuuint32_t estr[3] = {1, 1, 1};
        CUresult r = enc(&maps.m[k], CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, (void*)d_B, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        KB_REQUIRE(r == CUDA_SUCCESS, KBMOD_ERR_CUDA, "cuTensorMapEncodeTiled failed with %d (pitch %d)", (int)r,
                   PR_TW + 16 * k);
    }

    // ---- launches
    {
        const size_t n = (size_t)T * H * Wp;
        bound_plane_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(reinterpret_cast<const float2*>(d_psiphi), d_B, W,
                                                                        (int)Wp, (size_t)T * H);
    }
    int dev = 0, n_sm = 0;
    KB_CUDA(cudaGetDevice(&dev));
    KB_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    const int n_tiles = ((W + PR_TW - 1) / PR_TW) * ((H + PR_TH - 1) / PR_TH);
    const int grid = std::min(n_sm, n_tiles);
    PrunedTables tb{d_gvel, d_ge, d_offs, ng};
    KB_DISPATCH_TP(TPv, {
        KB_CUDA(cudaFuncSetAttribute(search_pruned_kernel<TP>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)PR_SMEM_BYTES));
        search_pruned_kernel<TP><<<grid, PR_THREADS, PR_SMEM_BYTES, st>>>(maps, reinterpret_cast<const float2*>(d_psiphi), T,
                                                                         H, W, d_tab, tb, P, bp, d_keys, d_stats);
        const size_t total = (size_t)H * W * P.K;
        finalize_kernel<TP><<<(unsigned)((total + FIN_THREADS - 1) / FIN_THREADS), FIN_THREADS,
                              (size_t)TP * FIN_THREADS * sizeof(float), st>>>(d_keys, reinterpret_cast<const float2*>(d_psiphi),
                                                                             H, W, d_tab, P, d_lh, d_flux, d_vel, d_nobs);
    });
    KB_CUDA(cudaGetLastError());
    if (n_launches) *n_launches = 3;
    return KBMOD_OK;
}
