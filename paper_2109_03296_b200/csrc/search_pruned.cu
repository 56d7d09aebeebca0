// (a3)-(a5) pruned search.  Same results as search_direct.cu; the full sigma-G evaluation runs only
// for trajectories whose EXACT upper bound reaches the threshold min_lh (trajectories
// with a recomputed likelihood below 10 are rejected; L115: only sum-LH > 10 leave the GPU).
//
// Bound.  For any kept set S the sigma-G filter can produce,
//     L' = sum_S psi / sqrt(sum_S phi)  <=  sum_valid max(psi, 0) / sqrt(F(m(n) - n_low))  =: U
// because sum_S psi <= sum_valid psi_+, and S always contains every sample between the two percentiles (the clip
// window is the median +- n_sigma*C*(P_hi - P_lo) with n_sigma*C >= 1 and P_lo <= P_50 <= P_hi), so |S| >= m(n);
// at most n_low members of S have phi below their epoch's floor f_t, the others have phi >= f_t, and F(k) is the
// sum of the k smallest floors.  U needs ONE packed 32-bit word per trajectory-epoch evaluation:
//     word = ceil(psi_+ / unit) << 2c  |  (phi < f_t) << c  |  1        (c = bits of an epoch count; 0 = invalid)
// so a single integer add per evaluation accumulates the fixed-point sum (rounded up), n_low and n.
//
// Kernels (all on the caller's stream, per batch of tiles):
//   bound_scale_kernel   once: per-epoch floors, the fixed-point unit and the thresholds thr[k]
//   bound_plane_kernel   once: the packed planes, row pitch a multiple of 4 so that TMA boxes start 16-byte aligned
//   bound_phase_kernel   where the time goes.  Persistent, one CTA per SM = 16 consumer warps + 1 producer warp
//                        group.  A CTA takes (64x32 tile of start pixels, 8 velocity groups) work units from a global
//                        counter; a group is <= 16 velocities adjacent in displacement space.  For each epoch the
//                        tile (+) the group's displacement bounding box is staged by TMA (zero fill outside the
//                        image = the off-chip rule) into a byte ring in shared memory, up to 16 regions ahead, and
//                        every consumer thread gathers its 4 pixels x 16 velocities from it: 4 B per
//                        trajectory-epoch evaluation, one conflict-free LDS.32 and one integer add.  full/empty
//                        mbarriers per in-flight region; no CTA-wide barrier anywhere in the loop.  (pixel,
//                        velocity) pairs whose bound reaches min_lh are appended to a global queue.
//   exact_queue_kernel   the queued pairs get the same evaluation as the direct kernel (8-byte gathers from the
//                        padded canvas, register sorting network); results enter the per-pixel top-K through a
//                        cascade of 64-bit atomicMax on (orderable L', ~vel_idx) keys.
//   exact_overflow_kernel  (tile, group, warp) items that did not fit the queue, all pairs evaluated.
// search_common.cu's finalize_kernel turns the keys into the four output arrays.
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "common.cuh"
#include "tma.cuh"

namespace {

constexpr int PR_TW = 64, PR_TH = 32;      // tile of start pixels per CTA
constexpr int PR_PIX = (PR_TW / 32) * (PR_TH / 16);  // pixels per consumer thread: (x + 32 h, y + 16 v), index 2 v + h
constexpr int PR_G = 16;                   // velocities per group
constexpr int PR_CONSUMERS = 512;          // 16 warps; thread = (x, y) and (x+32, y)
constexpr int PR_THREADS = PR_CONSUMERS + 128;  // + the producer warp group (one of its threads works)
constexpr int PR_RB = 8;                   // rows per TMA box
constexpr int PR_NPITCH = 12;              // tensor maps: pitch = 64 + 16*k elements, k < 12  (<= 240)
constexpr int PR_NHEIGHT = 4;              // ... x box heights of 8, 16, 32, 64 rows: a region is a few boxes
#ifndef KB_NB
#define KB_NB 16
#endif
constexpr int PR_NB = KB_NB;               // regions in flight (mbarrier pairs); a power of two
constexpr int PR_NTBL = 4;                 // group tables in flight
constexpr int PR_SMEM_MAX = 232448;        // 227 KB: the opt-in maximum of dynamic shared memory per CTA
constexpr int PR_SMEM_MISC = 512;          // barriers + producer bookkeeping
static_assert(PR_NB * 16 + 16 + 8 + PR_NB * 4 <= PR_SMEM_MISC, "full/empty barriers, unit mailbox and footprints must fit");
static_assert((PR_NB & (PR_NB - 1)) == 0, "PR_NB must be a power of two");
constexpr int PR_WAVES_PER_BATCH = 7;
#ifndef KB_SUB
#define KB_SUB 8
#endif
constexpr int PR_SUB = KB_SUB;                  // groups per work unit: CTAs take (tile, PR_SUB groups) units dynamically
// 20 warps = 5 per scheduler: 16384 registers / (5 x 32) = 102 -> 96 per thread at launch.  setmaxnreg moves
// registers inside the CTA's own allocation (640 x 96 = 61440): the producer warp group drops to 24 and the
// 16 consumer warps rise (512 x 104 + 128 x 56 = 60416 <= 61440)
constexpr int PR_REGS_PRODUCER = 56, PR_REGS_CONSUMER = 104;      // tiles per batch = SMs x this (the queue is reused per batch)

// per (group, epoch): where the staged region comes from and where it goes in the ring
struct __align__(16) GroupEpoch {
    int32_t ox, oy;       // region origin relative to the tile origin (min dx rounded down to even, min dy)
    uint16_t pitch_k;     // low byte: tensor map / pitch index (pitch = PR_TW + 16 * k elements); bit 8: every
                          // velocity of the group has the same displacement at this epoch ("uniform")
    uint16_t n_box;       // boxes of PR_RB rows
    uint32_t smem_off;    // byte offset of the region in the ring (the chain restarts at 0 for every tile)
    uint32_t footprint;   // ring bytes charged to this region = its size + the unused tail skipped before it
    uint32_t vmask;       // bit j: velocity slot j of the group is in use
    uint32_t pad_[2];
};
static_assert(sizeof(GroupEpoch) == 32, "GroupEpoch must be 32 bytes");

// table block of one group, copied to shared memory with the group's first region:
//   int32 offs[T][PR_G] (element offset of velocity j's displacement inside the region), GroupEpoch ge[T]
__host__ __device__ inline int tbl_bytes(int T) { return T * (PR_G * 4 + (int)sizeof(GroupEpoch)); }

struct PrunedTables {  // device pointers into the workspace
    const int32_t* gvel;          // [n_groups][PR_G]  velocity index or -1
    const unsigned char* gtbl;    // [n_groups] table blocks of tbl_bytes(T)
    // bit t of maskx[g][tile column] & masky[g][tile row]: the staged region of (tile, group g, epoch t) touches the
    // image.  Where it does not, every sample of the tile's trajectories is off-chip: the epoch is skipped, and the
    // whole group when fewer than min_obs epochs are left
    const unsigned long long* maskx;  // [n_groups][tiles_x]
    const unsigned long long* masky;  // [n_groups][tiles_y]
    const uint32_t* gfoot;        // [n_groups] ring bytes of all the regions of a group (charged when it is skipped)
    int n_groups;
    int ring_bytes;
};

struct TensorMaps {
    CUtensorMap m[PR_NHEIGHT * PR_NPITCH];  // [height code][pitch index]
};

struct BoundParams {
    unsigned char mkept[KBMOD_MAX_T + 1];  // m(n)
    int mk_min;                            // min of m(n) over n >= max(1, min_obs): what the quick group test may count on
    int pass_all;                          // min_lh <= 0 (or not finite): nothing can be pruned
    int cbits;                             // width of the two count fields of a plane word: 2^cbits > T
};

// device-side scalars and tables of the fixed-point planes, written by bound_scale_kernel (floats)
constexpr int SC_UNIT = 0, SC_INV_UNIT = 1, SC_CAP = 2, SC_FLOOR = 4, SC_THR = SC_FLOOR + KBMOD_MAX_T,
              SC_FLOATS = SC_THR + KBMOD_MAX_T + 1;

// threshold table of the bound test: indexed by the low 2 cbits bits of an accumulator (n_low << cbits | n_valid), holds
// the smallest accumulator value that passes; behind the scale table in the scratch
constexpr size_t TT_BYTES = 4u << (2 * 7);                    // KBMOD_MAX_T = 64 -> cbits = 7

struct Queue {
    uint2* entries;                  // (pixel index y0*W+x0, velocity index); v = 0xFFFFFFFF: hole
    unsigned long long* count;       // entries appended (may exceed cap: the excess overflowed)
    unsigned long long* units;       // work units handed out to the CTAs of the running launch (count + 1)
    unsigned long long cap;
    unsigned int* overflow;          // bitmap over (tile, group, warp) items that did not fit
};

// ---------------------------------------------------------------------------------------------
// bound planes: one 32-bit word per pixel, 0 for invalid pixels (and outside the image, by TMA zero fill);
// row pitch Wp (a multiple of 4 so that TMA boxes start 16-byte aligned).  With c = cbits, for a valid pixel
//     word = ceil(psi_+ / unit) << 2c  |  (phi < f_t) << c  |  1
// so that ONE integer add per trajectory-epoch accumulates the fixed-point sum of psi_+ (rounded up), the number
// of "low" samples and the number of valid samples.  f_t = the floor of epoch t: the largest of the candidates
// (0.40 + 0.02 k) x mean_t(phi) that at most 3 % of a sample of the epoch's valid pixels fall below.
// A kept set S has at least m(n) members, at most n_low of them low, and the others have phi >= f_t of their
// epoch, so  sum_S phi >= F(m(n) - n_low),  F(k) = the sum of the k smallest floors of the stack, and
//     L' <= sum psi_+ / sqrt(F(m(n) - n_low)).
// In units: pass iff sum >= thr[k] = THR sqrt(F(k) / f_min), unit = min_lh sqrt(f_min) / THR.  A term is clamped
// to `cap` units (T terms stay inside the sum field) and THR is chosen so that thr[k] <= 0.98 cap for every k:
// a clamped term passes on its own.  Any floors > 0 and any unit > 0 give a CORRECT bound; these make it tight.
constexpr int SC_BINS = 40, SC_SAMPLES = 16384;
__global__ void __launch_bounds__(1024)
bound_scale_kernel(const float2* __restrict__ psiphi, int T, int H, int W, float min_lh,
                                   const __grid_constant__ BoundParams BP, int need, float* __restrict__ scale,
                                   unsigned int* __restrict__ thrtab) {
    __shared__ float ssum[32];
    __shared__ int scnt[32];
    __shared__ int hist[SC_BINS + 1];
    __shared__ float s_mean;
    __shared__ float floors[KBMOD_MAX_T];
    const size_t plane = (size_t)H * W;
    const size_t n_samp = plane < SC_SAMPLES ? plane : SC_SAMPLES;
    // the stride is made coprime with the row length, so that the samples spread over every column and row instead
    // of landing in a handful of columns (a bad column or a masked disc would bias the floors)
    size_t stride = plane / n_samp;
    if (stride > 1) {
        stride = (stride - 1) | 1;  // odd and not larger than before: (n_samp - 1) * stride stays inside the plane
        for (;;) {
            size_t a = stride, b = (size_t)W;
            while (b) { const size_t r = a % b; a = b; b = r; }
            if (a == 1) break;
            stride -= 2;
        }
    }
    for (int t = 0; t < T; ++t) {
        const float2* pl = psiphi + (size_t)t * plane;
        float sum = 0.0f;
        int cnt = 0;
        for (size_t k = threadIdx.x; k < n_samp; k += blockDim.x) {
            const float phi = __ldg(pl + k * stride).y;
            if (phi > 0.0f && phi < CUDART_INF_F) { sum += phi; ++cnt; }
        }
        for (int d = 16; d > 0; d >>= 1) {
            sum += __shfl_down_sync(0xFFFFFFFFu, sum, d);
            cnt += __shfl_down_sync(0xFFFFFFFFu, cnt, d);
        }
        __syncthreads();  // the previous epoch's hist / s_mean are no longer read
        if ((threadIdx.x & 31) == 0) { ssum[threadIdx.x >> 5] = sum; scnt[threadIdx.x >> 5] = cnt; }
        if (threadIdx.x <= SC_BINS) hist[threadIdx.x] = 0;
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { sum += ssum[w]; cnt += scnt[w]; }
            scnt[0] = cnt;
            s_mean = cnt > 0 ? sum / (float)cnt : 0.0f;
        }
        __syncthreads();
        const float mean = s_mean;
        const bool usable = mean > 0.0f && mean < CUDART_INF_F;
        if (usable) {
            for (size_t k = threadIdx.x; k < n_samp; k += blockDim.x) {
                const float phi = __ldg(pl + k * stride).y;
                if (phi > 0.0f && phi < CUDART_INF_F) {
                    const float r = (phi / mean - 0.40f) * 50.0f;  // bin 1 + k holds [0.40 + 0.02 k, 0.40 + 0.02 (k+1))
                    const int bin = r < 0.0f ? 0 : (r >= (float)(SC_BINS - 1) ? SC_BINS : 1 + (int)r);
                    atomicAdd(&hist[bin], 1);  // bin 0: below 0.40 x mean
                }
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            float f = 0.0f;  // 0: this epoch has no usable sample; it gets the smallest floor of the others
            if (usable) {
                const int budget = (int)(0.03f * (float)scnt[0]);
                int below = hist[0], k = 0;  // below = samples under 0.40 + 0.02 k
                while (k + 1 < SC_BINS && below + hist[k + 1] <= budget) { below += hist[k + 1]; ++k; }
                f = (0.40f + 0.02f * (float)k) * mean;
                if (!(f > 1e-30f) || !(f < 1e30f)) f = 0.0f;
            }
            floors[t] = f;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        float fmin = CUDART_INF_F;
        for (int t = 0; t < T; ++t)
            if (floors[t] > 0.0f) fmin = fminf(fmin, floors[t]);
        if (!(fmin < CUDART_INF_F)) fmin = 1.0f;
        for (int t = 0; t < T; ++t) {
            if (!(floors[t] > 0.0f)) floors[t] = fmin;
            scale[SC_FLOOR + t] = floors[t];
        }
        // F(k): sum of the k smallest floors (insertion sort, T <= 64)
        for (int i = 1; i < T; ++i) {
            const float key = floors[i];
            int j = i - 1;
            while (j >= 0 && floors[j] > key) { floors[j + 1] = floors[j]; --j; }
            floors[j + 1] = key;
        }
        float Fk = 0.0f, ratio[KBMOD_MAX_T + 1];
        ratio[0] = 0.0f;
        for (int k = 1; k <= KBMOD_MAX_T; ++k) {
            if (k <= T) Fk += floors[k - 1] * 0.999999f;  // rounded down
            ratio[k] = sqrtf(Fk / fmin);
        }
        const int sum_bits = 32 - 2 * BP.cbits;
        // the largest term value: T of them must stay inside the sum field.  0.999: 2^sum_bits - 1 is not a float32
        // (it would round UP to 2^sum_bits and T clamped terms would wrap the field)
        const float cap = floorf(0.999f * (float)(1u << sum_bits) / (float)T);
        const float thr_units = 0.98f * cap / fmaxf(ratio[T], 1.0f);
        const float ml = (min_lh > 0.0f && min_lh < CUDART_INF_F) ? min_lh : 1.0f;
        float unit = ml * sqrtf(fmin) / thr_units;
        if (!(unit > 1e-30f) || !(unit < 1e30f)) unit = 1.0f;
        scale[SC_UNIT] = unit;
        scale[SC_INV_UNIT] = 1.0f / unit;
        scale[SC_CAP] = cap;
        // U = sum * unit / sqrt(F(k)) >= min_lh  <=>  sum >= thr_units * sqrt(F(k) / fmin); slack for float32 rounding
        for (int k = 0; k <= KBMOD_MAX_T; ++k) scale[SC_THR + k] = thr_units * ratio[k] * (1.0f - 1e-4f);
        scale[SC_THR] = 0.0f;  // no epoch is known to have phi >= its floor: no bound, always pass
    }
    __syncthreads();
    // The bound test as one table lookup.  An accumulator is  sum << 2c | n_low << c | n;  entry [n_low << c | n] is
    // the smallest accumulator that passes: ceil(thr[max(m(n) - n_low, 0)]) << 2c (the float test
    // (float)sum >= thr is sum >= ceil(thr) for an integer sum), 0 = always (no bound), ~0 = never (n < need).
    const unsigned int cmask = (1u << BP.cbits) - 1u;
    for (unsigned int idx = threadIdx.x; idx < (1u << (2 * BP.cbits)); idx += blockDim.x) {
        const int n = (int)(idx & cmask), n_low = (int)(idx >> BP.cbits);
        unsigned int e;
        if (n < need || n > T) e = 0xFFFFFFFFu;
        else if (BP.pass_all) e = 0u;
        else {
            const int m_eff = max((int)BP.mkept[n] - n_low, 0);
            const float th = scale[SC_THR + m_eff];
            e = th <= 0.0f ? 0u : ((unsigned int)ceilf(th)) << (2 * BP.cbits);
        }
        thrtab[idx] = e;
    }
}

__global__ void bound_plane_kernel(const float2* __restrict__ psiphi, unsigned int* __restrict__ B, int H, int W, int Wp,
                                   size_t rows /* T*H */, int cbits, const float* __restrict__ scale) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows * (size_t)Wp) return;
    const size_t r = i / Wp;
    const int x = (int)(i - r * Wp);
    unsigned int o = 0u;
    if (x < W) {
        const float2 s = __ldg(psiphi + r * W + x);
        if (s.y > 0.0f) {
            // rounded up twice over: the factor covers the float32 product, ceilf the quantisation
            const float t = fmaxf(s.x, 0.0f) * __ldg(scale + SC_INV_UNIT) * 1.000001f;
            const float cap = __ldg(scale + SC_CAP);
            const unsigned int fix = (t < cap) ? (unsigned int)ceilf(t) : (unsigned int)cap;  // inf, too
            const unsigned int low = (s.y < __ldg(scale + SC_FLOOR + (int)(r / (size_t)H))) ? 1u : 0u;
            o = (fix << (2 * cbits)) | (low << cbits) | 1u;
        }
    }
    B[i] = o;
}

// insert into a descending list of K keys shared by all CTAs (empty = 0): each slot ends up
// holding the maximum of everything that reached it, so the list is the top-K of all insertions.
__device__ __forceinline__ void topk_insert(unsigned long long* keys, int K, unsigned long long key) {
    for (int k = 0; k < K && key != 0ull; ++k) {
        const unsigned long long old = atomicMax(keys + k, key);
        key = old < key ? old : key;  // whichever lost moves on to the next slot
    }
}

__device__ __forceinline__ void tile_origin(int tile_lin, int tiles_x, int tiles_y, int& tile_x0, int& tile_y0, int& txi_out,
                                            int& tyi_out) {
    // column-block order: 4 tile columns x all tile rows, then the next 4 columns, so that the CTAs
    // running at the same time work on a compact block of tiles and share their staged regions in L2
    const int cb = tile_lin / (4 * tiles_y), rem = tile_lin - cb * 4 * tiles_y;
    const int cols_here = min(4, tiles_x - cb * 4);
    const int tyi = rem / cols_here, txi = cb * 4 + rem - tyi * cols_here;
    tile_x0 = txi * PR_TW;
    tile_y0 = tyi * PR_TH;
    txi_out = txi;
    tyi_out = tyi;
}
__device__ __forceinline__ void tile_origin(int tile_lin, int tiles_x, int tiles_y, int& tile_x0, int& tile_y0) {
    int a, b;
    tile_origin(tile_lin, tiles_x, tiles_y, tile_x0, tile_y0, a, b);
}

// ---------------------------------------------------------------------------------------------
// phase 1: bounds from shared-memory tiles; survivors -> queue
__global__ void __launch_bounds__(PR_THREADS, 1)
bound_phase_kernel(const __grid_constant__ TensorMaps maps, int T, int row_begin, int row_end, int W, int tile_begin,
                   int tile_end, int g_begin, int g_end,
                   const __grid_constant__ PrunedTables tb, const __grid_constant__ BoundParams BP, int min_obs,
                   const unsigned int* __restrict__ thrtab, const __grid_constant__ Queue Qu) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const int TBL = tbl_bytes(T);
    unsigned char* tblbase = smem + tb.ring_bytes;
    uint64_t* full = reinterpret_cast<uint64_t*>(tblbase + PR_NTBL * TBL);
    uint64_t* empty = full + PR_NB;
    uint64_t* ufull = empty + PR_NB;   // work-unit mailbox: the producer takes a unit from the global counter and
    uint64_t* uempty = ufull + 1;      // publishes its index here; the consumers acknowledge having read it
    volatile uint32_t* mailbox = reinterpret_cast<volatile uint32_t*>(uempty + 1);
    uint32_t* fpq = reinterpret_cast<uint32_t*>(uempty + 2);  // producer only: footprint of each region in flight

    const int tid = threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        for (int i = 0; i < PR_NB; ++i) {
            kb_mbar_init(&full[i], 1);
            kb_mbar_init(&empty[i], PR_CONSUMERS / 32);
        }
        kb_mbar_init(ufull, 1);
        kb_mbar_init(uempty, PR_CONSUMERS / 32);
        kb_fence_barrier_init();
        for (int k = 0; k < PR_NHEIGHT * PR_NPITCH; ++k) kb_prefetch_tensormap(&maps.m[k]);
    }
    __syncthreads();

    // tiles cover the band of start rows [row_begin, row_end): tile row r starts at image row row_begin + r * PR_TH
    const int tiles_x = (W + PR_TW - 1) / PR_TW, tiles_y = (row_end - row_begin + PR_TH - 1) / PR_TH;
    const int ng = tb.n_groups;
    // work units: (tile of the batch) x (PR_SUB consecutive groups of the chunk), tile-major
    const int n_sub = (g_end - g_begin + PR_SUB - 1) / PR_SUB;
    const unsigned int n_units = (unsigned int)(tile_end - tile_begin) * (unsigned int)n_sub;

    if (warp >= PR_CONSUMERS / 32) {
        // ------------------------------------------------------------------ producer (one thread)
        kb_reg_dec<PR_REGS_PRODUCER>();
        if (tid != PR_CONSUMERS) return;
        uint32_t q = 0, oldest = 0, used = 0, gcount = 0, carry = 0;
        uint32_t qs0 = 0, qs1 = 0, qs2 = 0, qs3 = 0;  // first region of the last four groups
        const uint32_t ring = (uint32_t)tb.ring_bytes;
        const int need = min_obs > 1 ? min_obs : 1;
        int4 nxt0 = make_int4(0, 0, 0, 0);
        uint32_t nxt_fp = 0;
        int nxt_g = -1;  // the group nxt0 / nxt_fp belong to
        for (uint32_t uk = 0;; ++uk) {
            if (uk > 0) kb_mbar_wait(uempty, (uk - 1) & 1);  // every consumer warp has read the previous unit
            const unsigned int u = (unsigned int)atomicAdd(Qu.units, 1ull);
            *mailbox = u;
            kb_mbar_arrive(ufull);
            if (u >= n_units) break;
            const int tile_lin = tile_begin + (int)(u / (unsigned int)n_sub);
            const int g_lo = g_begin + (int)(u % (unsigned int)n_sub) * PR_SUB, g_hi = min(g_end, g_lo + PR_SUB);
            int tile_x0, tile_y0, txi, tyi;
            tile_origin(tile_lin, tiles_x, tiles_y, tile_x0, tile_y0, txi, tyi);
            tile_y0 += row_begin;
            // the ring chain of the tables restarts at offset 0 for every unit: drain first
            while (oldest < q) {
                kb_mbar_wait(&empty[oldest & (PR_NB - 1)], (oldest / PR_NB) & 1);
                ++oldest;
            }
            used = 0;
            carry = 0;
            for (int g = g_lo; g < g_hi; ++g) {
                const unsigned long long on = __ldg(tb.maskx + (size_t)g * tiles_x + txi) & __ldg(tb.masky + (size_t)g * tiles_y + tyi);
                if (__popcll(on) < need) {  // no trajectory of this tile and group can have min_obs valid epochs
                    carry += __ldg(tb.gfoot + g);
                    continue;
                }
                qs0 = qs1; qs1 = qs2; qs2 = qs3; qs3 = q;
                const unsigned char* gt = tb.gtbl + (size_t)g * TBL;
                const GroupEpoch* gge = reinterpret_cast<const GroupEpoch*>(gt + (size_t)T * PR_G * 4);
                // the first epoch's entry was fetched from global memory one group ago (nxt0 / nxt_fp); the other
                // epochs are read from the group's table in shared memory once it has landed: no global-memory
                // latency on the producer's critical path
                if (nxt_g != g) {
                    nxt0 = __ldg(reinterpret_cast<const int4*>(gge));
                    nxt_fp = __ldg(&gge->footprint);
                }
                int4 e0 = nxt0;
                uint32_t fp = nxt_fp;
                const unsigned char* tblp = tblbase + (gcount & (PR_NTBL - 1)) * TBL;
                const GroupEpoch* sge = reinterpret_cast<const GroupEpoch*>(tblp + (size_t)T * PR_G * 4);
                const uint32_t q_first = q;
                bool tbl_landed = false;
                for (int t = 0; t < T; ++t) {  // epoch 0 has no displacement: its region is the tile, always on the image
                    if (t >= 1) {
                        if (!tbl_landed) {
                            kb_mbar_wait(&full[q_first & (PR_NB - 1)], (q_first / PR_NB) & 1);  // the table is in
                            tbl_landed = true;
                        }
                        fp = sge[t].footprint;
                        if (!((on >> t) & 1ull)) {  // skipped: its ring bytes are charged to the next staged region
                            carry += fp;
                            continue;
                        }
                        e0 = *reinterpret_cast<const int4*>(sge + t);
                    }
                    const int pitch_k = e0.z & 0xFF, n_box = (unsigned)e0.z >> 16;
                    if (carry + fp > ring / 2) {
                        // a long run of skipped regions: rather than charge it, wait until nothing is in flight
                        while (oldest < q) {
                            kb_mbar_wait(&empty[oldest & (PR_NB - 1)], (oldest / PR_NB) & 1);
                            ++oldest;
                        }
                        used = 0;
                        carry = 0;
                    }
                    fp += carry;
                    carry = 0;
                    // table slot gcount & 3 was last read by group gcount - 4: all its regions must be released
                    const bool tbl_busy_possible = (t == 0) && gcount >= PR_NTBL;
                    while (used + fp > ring || q - oldest >= PR_NB || (tbl_busy_possible && oldest < qs0)) {
                        kb_mbar_wait(&empty[oldest & (PR_NB - 1)], (oldest / PR_NB) & 1);
                        used -= fpq[oldest & (PR_NB - 1)];
                        ++oldest;
                    }
                    const int slot = q & (PR_NB - 1);
                    fpq[slot] = fp;
                    used += fp;
                    const int pitch = PR_TW + 16 * pitch_k;
                    const uint32_t box_bytes = (uint32_t)pitch * PR_RB * sizeof(unsigned int);
                    kb_mbar_expect_tx(&full[slot], box_bytes * n_box + (t == 0 ? (uint32_t)TBL : 0u));
                    if (t == 0) kb_bulk_load_1d(tblbase + (gcount & (PR_NTBL - 1)) * TBL, gt, (uint32_t)TBL, &full[slot]);
                    unsigned char* dst = smem + (uint32_t)e0.w;
                    // the region's rows (a multiple of 8) as the fewest boxes of 64, 32, 16 or 8 rows: the producer is a
                    // single thread and every instruction it issues competes with four busy consumer warps
                    int left = n_box, done = 0;
                    while (left > 0) {
                        const int hc = left >= 8 ? 3 : (left >= 4 ? 2 : (left >= 2 ? 1 : 0));
                        kb_tma_load_3d(dst + (size_t)done * box_bytes, &maps.m[hc * PR_NPITCH + pitch_k], tile_x0 + e0.x,
                                       tile_y0 + e0.y + done * PR_RB, t, &full[slot]);
                        done += 1 << hc;
                        left -= 1 << hc;
                    }
                    ++q;
                    if (t == 0) {  // fetch the next group's first entry now: a whole group of time to arrive
                        nxt_g = (g + 1 < g_hi) ? g + 1 : -1;
                        if (nxt_g >= 0) {
                            const GroupEpoch* nge = reinterpret_cast<const GroupEpoch*>(tb.gtbl + (size_t)nxt_g * TBL + (size_t)T * PR_G * 4);
                            nxt0 = __ldg(reinterpret_cast<const int4*>(nge));
                            nxt_fp = __ldg(&nge->footprint);
                        }
                    }
                }
                ++gcount;
            }
        }
        return;
    }

    // ---------------------------------------------------------------------- consumers
    kb_reg_inc<PR_REGS_CONSUMER>();
    const int need = min_obs > 1 ? min_obs : 1;
    uint32_t q = 0, gcount = 0;
    for (uint32_t uk = 0;; ++uk) {
        kb_mbar_wait(ufull, uk & 1);
        const unsigned int u = *mailbox;
        __syncwarp();
        if (lane == 0) kb_mbar_arrive(uempty);
        if (u >= n_units) break;
        const int tile_lin = tile_begin + (int)(u / (unsigned int)n_sub);
        const int g_lo = g_begin + (int)(u % (unsigned int)n_sub) * PR_SUB, g_hi = min(g_end, g_lo + PR_SUB);
        int tile_x0, tile_y0, txi, tyi;
        tile_origin(tile_lin, tiles_x, tiles_y, tile_x0, tile_y0, txi, tyi);
        tile_y0 += row_begin;
        const int px0 = tile_x0 + lane, py0 = tile_y0 + warp;  // this thread's pixels: (px0 + 32 h, py0 + 16 v)

        for (int g = g_lo; g < g_hi; ++g) {
            // epochs whose staged region touches the image (the same test as the producer's)
            const unsigned long long on = __ldg(tb.maskx + (size_t)g * tiles_x + txi) & __ldg(tb.masky + (size_t)g * tiles_y + tyi);
            if (__popcll(on) < need) continue;
            const unsigned char* tblp = tblbase + (gcount & (PR_NTBL - 1)) * TBL;
            ++gcount;
            const int4* offs4 = reinterpret_cast<const int4*>(tblp);
            const GroupEpoch* ge = reinterpret_cast<const GroupEpoch*>(tblp + (size_t)T * PR_G * 4);
            // per (pixel, velocity): fixed-point sum of psi_+ << 14 | low-phi samples << 7 | valid samples
            unsigned int AN[PR_PIX][PR_G];
#pragma unroll
            for (int j = 0; j < PR_G; ++j)
#pragma unroll
                for (int i = 0; i < PR_PIX; ++i) AN[i][j] = 0u;
            // epochs at which the whole group shares one displacement (the first night: a few pixels of motion)
            // are gathered once per pixel and folded into the 16 accumulators at the end
            unsigned int ANU[PR_PIX];
#pragma unroll
            for (int i = 0; i < PR_PIX; ++i) ANU[i] = 0u;
            unsigned long long rem = on;  // bit 0 is always set: epoch 0 has no displacement
#pragma unroll 1
            while (rem) {
                const int t = __ffsll((long long)rem) - 1;
                rem &= rem - 1;
                const int slot = q & (PR_NB - 1);
                kb_mbar_wait(&full[slot], (q / PR_NB) & 1);  // (the group's tables came with the region of epoch 0)
                const uint2 cur = *reinterpret_cast<const uint2*>(&ge[t].pitch_k);  // {pitch_k | uniform << 8 | n_box << 16, smem_off}
                const int pitch = PR_TW + 16 * (int)(cur.x & 0xFFu);
                const unsigned char* base = smem + cur.y + (size_t)(warp * pitch + lane) * sizeof(unsigned int);
                const int rows16 = 16 * pitch * (int)sizeof(unsigned int);  // this thread's second row of pixels
                if (cur.x & 0x100u) {
                    const unsigned char* p = base + offs4[t * (PR_G / 4)].x;
#pragma unroll
                    for (int v = 0; v < PR_TH / 16; ++v) {
                        const unsigned int* pv = reinterpret_cast<const unsigned int*>(p + v * rows16);
                        ANU[2 * v] += pv[0];
                        ANU[2 * v + 1] += pv[32];
                    }
                } else {
                    // two non-uniform epochs at a time: one three-operand add takes both words
                    const int t2 = rem ? __ffsll((long long)rem) - 1 : -1;
                    const uint2 cur2 = (t2 >= 0) ? *reinterpret_cast<const uint2*>(&ge[t2].pitch_k) : make_uint2(0x100u, 0u);
                    // ... if the second region has landed already: waiting for it while holding the first could
                    // deadlock against the producer waiting for ring space (lane 0 decides for the warp)
                    const int slot2 = (q + 1) & (PR_NB - 1);
                    const bool both = !(cur2.x & 0x100u) &&
                                      __shfl_sync(0xFFFFFFFFu, (int)kb_mbar_test(&full[slot2], ((q + 1) / PR_NB) & 1), 0) != 0;
                    if (both) {
                        rem &= rem - 1;
                        kb_mbar_wait(&full[slot2], ((q + 1) / PR_NB) & 1);  // completed: acquires it for every lane
                        const int pitch2 = PR_TW + 16 * (int)(cur2.x & 0xFFu);
                        const unsigned char* base2 = smem + cur2.y + (size_t)(warp * pitch2 + lane) * sizeof(unsigned int);
                        const int rows16b = 16 * pitch2 * (int)sizeof(unsigned int);
#pragma unroll
                        for (int k = 0; k < PR_G / 4; ++k) {
                            const int4 o = offs4[t * (PR_G / 4) + k], o2 = offs4[t2 * (PR_G / 4) + k];
                            const int oo[4] = {o.x, o.y, o.z, o.w}, oo2[4] = {o2.x, o2.y, o2.z, o2.w};
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                const unsigned char* p = base + oo[i];
                                const unsigned char* p2 = base2 + oo2[i];
#pragma unroll
                                for (int v = 0; v < PR_TH / 16; ++v) {
                                    const unsigned int* pv = reinterpret_cast<const unsigned int*>(p + v * rows16);
                                    const unsigned int* pv2 = reinterpret_cast<const unsigned int*>(p2 + v * rows16b);
                                    AN[2 * v][4 * k + i] += pv[0] + pv2[0];
                                    AN[2 * v + 1][4 * k + i] += pv[32] + pv2[32];
                                }
                            }
                        }
                        __syncwarp();
                        if (lane == 0) {
                            kb_mbar_arrive(&empty[slot]);
                            kb_mbar_arrive(&empty[slot2]);
                        }
                        q += 2;
                        continue;
                    }
#pragma unroll
                    for (int k = 0; k < PR_G / 4; ++k) {
                        const int4 o = offs4[t * (PR_G / 4) + k];  // byte offsets inside the region
                        const int oo[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const unsigned char* p = base + oo[i];
#pragma unroll
                            for (int v = 0; v < PR_TH / 16; ++v) {
                                const unsigned int* pv = reinterpret_cast<const unsigned int*>(p + v * rows16);
                                AN[2 * v][4 * k + i] += pv[0];
                                AN[2 * v + 1][4 * k + i] += pv[32];
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) kb_mbar_arrive(&empty[slot]);  // this warp is done with the region
                ++q;
            }
            // ---- bound test; survivors -> queue
            unsigned int m[PR_PIX];
            const uint32_t vmask = __ldg(reinterpret_cast<const uint32_t*>(tb.gtbl + (size_t)g * TBL + (size_t)T * PR_G * 4 +
                                                                            offsetof(GroupEpoch, vmask)));
            int my_cnt = 0;
            // the bound test: one table lookup per (pixel, velocity), indexed by the accumulator's two count fields
            // (bound_scale_kernel; n < min_obs never passes)
            const unsigned int idx_mask = (1u << (2 * BP.cbits)) - 1u;
#pragma unroll
            for (int h = 0; h < PR_PIX; ++h) {
                const bool in_img = (px0 + 32 * (h & 1)) < W && (py0 + 16 * (h >> 1)) < row_end;
                m[h] = 0u;
#pragma unroll
                for (int j = 0; j < PR_G; ++j) {
                    const unsigned int an = AN[h][j] + ANU[h];
                    const unsigned int need_an = __ldg(thrtab + (an & idx_mask));
                    m[h] |= (an >= need_an ? 1u : 0u) << j;
                }
                m[h] = in_img ? (m[h] & vmask) : 0u;
                my_cnt += __popc(m[h]);
            }
            const int total = __reduce_add_sync(0xFFFFFFFFu, my_cnt);
            if (total > 0) {
                unsigned long long base = 0;
                if (lane == 0) base = atomicAdd(Qu.count, (unsigned long long)total);
                base = __shfl_sync(0xFFFFFFFFu, base, 0);
                if (base + (unsigned long long)total <= Qu.cap) {
                    // entries in (half, velocity, lane) order: neighbours in the queue are neighbouring pixels with
                    // the same velocity, so the exact kernel's gathers coalesce
                    unsigned long long pos = base;
                    const unsigned int pixlin = (unsigned int)(py0 * W + px0);
                    const unsigned int lt = (1u << lane) - 1u;
#pragma unroll
                    for (int h = 0; h < PR_PIX; ++h) {
                        unsigned int any = __reduce_or_sync(0xFFFFFFFFu, m[h]);
                        while (any) {
                            const int j = __ffs(any) - 1;
                            any &= any - 1;
                            const bool mine = (m[h] >> j) & 1u;
                            const unsigned int bal = __ballot_sync(0xFFFFFFFFu, mine);
                            if (mine) {
                                const int v = __ldg(tb.gvel + (size_t)g * PR_G + j);
                                Qu.entries[pos + __popc(bal & lt)] =
                                    make_uint2(pixlin + 32u * (h & 1) + 16u * (unsigned int)W * (h >> 1), (unsigned int)v);
                            }
                            pos += __popc(bal);
                        }
                    }
                } else {
                    // the queue is full: the whole (tile, group, warp) item goes to the overflow kernel;
                    // the part of the reservation that lies inside the queue becomes holes
                    const size_t item = ((size_t)tile_lin * ng + g) * (PR_CONSUMERS / 32) + warp;
                    if (lane == 0) atomicOr(Qu.overflow + (item >> 5), 1u << (item & 31));
                    for (unsigned long long i = base + lane; i < base + total && i < Qu.cap; i += 32)
                        Qu.entries[i] = make_uint2(0u, 0xFFFFFFFFu);
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// phase 2: exact evaluation (steps 1-3 of kbmod_search) of one (pixel, velocity) pair + top-K insertion
struct ExactArgs {
    const float2* S4;
    S4Geom G;
    const int* off;      // [n_vel][kb_tp4(TP)]
    int W, row_begin, row_end;
    unsigned long long* keys;  // [row_end - row_begin][W][K]
};

// (A two-pass form -- filter values first, psi/phi of the same elements re-read afterwards, 85 registers, 3 CTAs per
// SM -- was measured: the second reads are not L1 hits and the phase took twice as long.)
// Returns true iff the trajectory has a result with L' >= min_lh.
template <int TP>
__device__ __forceinline__ bool eval_pair(const ExactArgs& A, const DevParams& P, int x0, int y0, int v, float* scratch,
                                          int stride) {
    const unsigned int base = (unsigned int)(y0 + A.G.pyn) * (unsigned int)A.G.Wp + (unsigned int)(x0 + A.G.pxn);
    float f[TP], m[TP], sp, sf;
    int n;
    kb_gather_s4<TP>(A.S4, base, reinterpret_cast<const int4*>(A.off + (size_t)v * kb_tp4(TP)), f, m, n);
    const int nk = kb_score_s4<TP, false>(f, m, n, P, scratch, stride, sp, sf);
    if (nk > 0) {
        const float lh = kb_lh_of(sp, sf);
        if (lh >= P.min_lh) {
            topk_insert(A.keys + ((size_t)(y0 - A.row_begin) * A.W + x0) * P.K, P.K, kb_topk_key(lh, v));
            return true;
        }
    }
    return false;
}

#ifndef KB_EX_THREADS
#define KB_EX_THREADS 256
#endif
constexpr int EX_THREADS = KB_EX_THREADS;
#ifndef KB_EX_CTAS
#define KB_EX_CTAS 2
#endif
constexpr int EX_CTAS_PER_SM = KB_EX_CTAS;
#ifndef KB_EX_BIG_T
#define KB_EX_BIG_T 32
#endif
#ifndef KB_EX_BIG_THREADS
#define KB_EX_BIG_THREADS 256
#endif
// lightcurves longer than KB_EX_BIG_T epochs do not fit 128 registers (T = 50: 228 bytes spilled per thread): one CTA
// of 256 threads per SM and up to 255 registers instead.  The phase is not occupancy-bound, the spills
// cost: configs[3]'s exact phase 1147 -> 1062 ms (384 threads at 168 registers: 1068; 512 at 128, spilling: 1166)
template <int TP> struct ExCfg {
    static constexpr bool big = TP > KB_EX_BIG_T;
    static constexpr int ctas = big ? 1 : EX_CTAS_PER_SM;
    static constexpr int threads = big ? KB_EX_BIG_THREADS : EX_THREADS;
};

template <int TP>
__global__ void __launch_bounds__(ExCfg<TP>::threads, ExCfg<TP>::ctas)
exact_queue_kernel(const __grid_constant__ ExactArgs A, const __grid_constant__ DevParams P,
                   const __grid_constant__ Queue Qu, unsigned long long* __restrict__ stats) {
    extern __shared__ float scratch_all[];  // [TP][threads]
    const unsigned long long cnt = *Qu.count;
    const unsigned long long n = cnt < Qu.cap ? cnt : Qu.cap;
    unsigned long long done = 0, passed = 0;
    // the trip count is warp-uniform and every iteration ends in __syncwarp(): without it the lanes of a warp
    // drift apart after the first divergent top-K insertion and run the whole body one by one from then on
    // (measured: 3.7 active threads per instruction)
    // Chunks of EX_CHUNK x 32 consecutive entries are handed to the warps from a counter (zeroed with the queue
    // counters).  A static grid-stride split left the SMs idle for 19 % of the kernel's duration (ncu: sm__cycles_active
    // against elapsed) and the warps in flight far apart in the queue: 100.2 ms per search against 79.6 ms this way.
    // The next entry of a chunk is fetched one iteration ahead.
    constexpr int EX_CHUNK = 16;  // 2 / 4 / 8 / 16 groups of 32 per grab: 83.6 / 82.0 / 82.0 / 81.4 ms
    unsigned long long* next_chunk = Qu.units + 1;
    const unsigned int lane = threadIdx.x & 31u;
    const uint2 hole = make_uint2(0u, 0xFFFFFFFFu);
    for (;;) {
        unsigned long long c = 0;
        if (lane == 0) c = atomicAdd(next_chunk, 1ull);
        c = __shfl_sync(0xFFFFFFFFu, c, 0);
        const unsigned long long base = c * (unsigned long long)(32 * EX_CHUNK);
        if (base >= n) break;
        uint2 e_next = (base + lane < n) ? __ldg(Qu.entries + base + lane) : hole;
#pragma unroll 1
        for (int k = 0; k < EX_CHUNK; ++k) {
            const uint2 e = e_next;
            const unsigned long long i_next = base + (unsigned long long)(k + 1) * 32 + lane;
            e_next = (k + 1 < EX_CHUNK && i_next < n) ? __ldg(Qu.entries + i_next) : hole;
            if (e.y != 0xFFFFFFFFu) {
                const int y0 = (int)(e.x / (unsigned)A.W), x0 = (int)(e.x - (unsigned)y0 * (unsigned)A.W);
                passed += eval_pair<TP>(A, P, x0, y0, (int)e.y, scratch_all + threadIdx.x, ExCfg<TP>::threads) ? 1ull : 0ull;
                ++done;
            }
            __syncwarp();
        }
    }
    // statistics: trajectories fully evaluated, and how many of them reached min_lh (candidates before the top-K)
    for (int d = 16; d > 0; d >>= 1) {
        done += __shfl_down_sync(0xFFFFFFFFu, done, d);
        passed += __shfl_down_sync(0xFFFFFFFFu, passed, d);
    }
    if ((threadIdx.x & 31) == 0 && done) {
        atomicAdd(stats, done);
        if (passed) atomicAdd(stats + 4, passed);
    }
}

// items that did not fit the queue: every pair of the (tile, group, warp) item is evaluated
template <int TP>
__global__ void __launch_bounds__(EX_THREADS)
exact_overflow_kernel(const __grid_constant__ ExactArgs A, const __grid_constant__ DevParams P,
                      const unsigned int* __restrict__ overflow, size_t n_words, const int32_t* __restrict__ gvel, int ng,
                      unsigned long long* __restrict__ stats) {
    extern __shared__ float scratch_all[];
    const int lane = threadIdx.x & 31;
    const size_t warp_global = ((size_t)blockIdx.x * EX_THREADS + threadIdx.x) >> 5;
    const size_t n_warps = ((size_t)gridDim.x * EX_THREADS) >> 5;
    const int W = A.W;
    const int tiles_x = (W + PR_TW - 1) / PR_TW, tiles_y = (A.row_end - A.row_begin + PR_TH - 1) / PR_TH;
    unsigned long long done = 0, passed = 0;
    for (size_t w = warp_global; w < n_words; w += n_warps) {
        unsigned int bits = __ldg(overflow + w);
        while (bits) {
            const int b = __ffs(bits) - 1;
            bits &= bits - 1;
            const size_t item = w * 32 + b;
            const int row = (int)(item % (PR_CONSUMERS / 32));
            const size_t tg = item / (PR_CONSUMERS / 32);
            const int g = (int)(tg % ng), tile_lin = (int)(tg / ng);
            int tile_x0, tile_y0;
            tile_origin(tile_lin, tiles_x, tiles_y, tile_x0, tile_y0);
            for (int h = 0; h < PR_PIX; ++h) {
                const int x0 = tile_x0 + lane + 32 * (h & 1), y0 = A.row_begin + tile_y0 + row + 16 * (h >> 1);
                for (int j = 0; j < PR_G; ++j) {
                    const int v = __ldg(gvel + (size_t)g * PR_G + j);
                    if (v >= 0 && x0 < W && y0 < A.row_end) {
                        passed += eval_pair<TP>(A, P, x0, y0, v, scratch_all + threadIdx.x, EX_THREADS) ? 1ull : 0ull;
                        ++done;
                    }
                    __syncwarp();  // keep the warp converged (see exact_queue_kernel)
                }
            }
        }
    }
    for (int d = 16; d > 0; d >>= 1) {
        done += __shfl_down_sync(0xFFFFFFFFu, done, d);
        passed += __shfl_down_sync(0xFFFFFFFFu, passed, d);
    }
    if (lane == 0 && done) {
        atomicAdd(stats, done);
        if (passed) atomicAdd(stats + 4, passed);
    }
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
// times[0]; a group whose staged region would not fit half the ring is bisected further), the
// per-(group, epoch) staging geometry and the ring offsets
namespace {

struct Planner {
    int T, n_vel, ring_bytes, max_region;
    const int32_t *dx, *dy;  // [n_vel][T], clamped so that any |d| beyond every image size stays off-image
    std::vector<int> idx, px, py;
    std::vector<std::pair<int, int>> leaves;

    // staged bytes of velocities idx[lo..hi) at epoch t (and the geometry, if asked for)
    long long region(int lo, int hi, int t, GroupEpoch* e, int* x0_out, int* y0_out) const {
        int x0 = INT32_MAX, x1 = INT32_MIN, y0 = INT32_MAX, y1 = INT32_MIN;
        for (int i = lo; i < hi; ++i) {
            const int v = idx[i];
            const int ddx = dx[(size_t)v * T + t], ddy = dy[(size_t)v * T + t];
            x0 = std::min(x0, ddx); x1 = std::max(x1, ddx); y0 = std::min(y0, ddy); y1 = std::max(y1, ddy);
        }
        // TMA: the box must start on a 16-byte boundary, i.e. at a multiple of 4 in x for 4-byte elements (a
        // misaligned start raises an illegal-instruction fault on sm_100a); tile origins are multiples of 64
        x0 -= (x0 & 3);
        const long long bw = (long long)x1 - x0 + PR_TW, bh = (long long)y1 - y0 + PR_TH;
        const long long pk = (bw - PR_TW + 15) / 16, nb = (bh + PR_RB - 1) / PR_RB;
        if (pk >= PR_NPITCH) return -1;
        if (e) {
            e->ox = x0; e->oy = y0; e->pitch_k = (uint16_t)pk; e->n_box = (uint16_t)nb;
        }
        if (x0_out) { *x0_out = x0; *y0_out = y0; }
        return (PR_TW + 16 * pk) * PR_RB * nb * (long long)sizeof(unsigned int);
    }
    bool fits(int lo, int hi) const {
        for (int t = 0; t < T; ++t) {
            const long long b = region(lo, hi, t, nullptr, nullptr, nullptr);
            if (b < 0 || b > max_region) return false;
        }
        return true;
    }
    void split(int lo, int hi) {
        const int n = hi - lo;
        if (n <= PR_G && (n == 1 || fits(lo, hi))) {
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
        int half;
        if (n > PR_G) {
            const int ngr = (n + PR_G - 1) / PR_G;
            half = (ngr / 2) * PR_G;  // split at a multiple of the group size: all leaves but one are full
        } else {
            half = n / 2;
        }
        split(lo, lo + half);
        split(lo + half, hi);
    }
};

int ring_bytes_for(int T) { return ((PR_SMEM_MAX - PR_SMEM_MISC - PR_NTBL * tbl_bytes(T)) / 1024) * 1024; }
size_t max_groups(int n_vel) {
    const size_t full = ((size_t)n_vel + PR_G - 1) / PR_G;
    return std::min((size_t)n_vel, 2 * full + 16);
}
size_t queue_cap(int n_vel) {
    // test hook: KBMOD_B200_QUEUE_CAP=<entries> shrinks the survivor queue so that the overflow path runs
    if (const char* e = getenv("KBMOD_B200_QUEUE_CAP")) {
        const long long v = atoll(e);
        if (v > 0) return (size_t)std::max<long long>(64, v);
    }
    const double want = 1100.0 * PR_TW * PR_TH * (double)n_vel / 32.0;
    return (size_t)std::min(536870912.0, std::max(1048576.0, want));  // at most 2^29 entries = 4 GiB
}
size_t n_tiles_of(int n_rows, int W) { return (size_t)((W + PR_TW - 1) / PR_TW) * ((n_rows + PR_TH - 1) / PR_TH); }
size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }

struct ScratchLayout {
    size_t B, qentries, qcount, overflow, total, overflow_words;
};
ScratchLayout scratch_layout(int T, int H, int W, int n_rows, int n_vel) {
    ScratchLayout L;
    const size_t ngm = max_groups(n_vel), Wp = ((size_t)W + 3) & ~(size_t)3;
    size_t o = 0;
    L.B = o;        o += al256((size_t)T * H * Wp * 4);
    L.qentries = o; o += al256(queue_cap(n_vel) * 8);
    // queue counters, then the scale table, then the threshold table of the bound test (2^(2 cbits) words, cbits <= 7)
    L.qcount = o;   o += 256 + al256(SC_FLOATS * sizeof(float)) + TT_BYTES;
    L.overflow_words = (n_tiles_of(n_rows, W) * ngm * (PR_CONSUMERS / 32) + 31) / 32;
    L.overflow = o; o += al256(L.overflow_words * 4);
    L.total = o;
    return L;
}

}  // namespace

size_t kb_pruned_scratch_bytes(int T, int H, int W, int n_rows, int n_vel) {
    return scratch_layout(T, H, W, n_rows, n_vel).total;
}

// ---------------------------------------------------------------------------------------------
// the host plan: velocity groups, staging geometry of every (group, epoch), ring chain, on-image masks
int kb_pruned_plan_build(int T, int H, int W, int row_begin, int row_end, const int32_t* h_dx, const int32_t* h_dy,
                         int n_vel, PrunedPlan* out) {
    PrunedPlan& PC = *out;
    PC = PrunedPlan();
    const int TBL = tbl_bytes(T);
    // displacements as the staging sees them: anything beyond every possible image size is off-image for all start
    // pixels, wherever exactly it is; clamping keeps the geometry inside int32 / TMA coordinates
    std::vector<int32_t> cdx((size_t)n_vel * T), cdy((size_t)n_vel * T);
    for (size_t i = 0; i < cdx.size(); ++i) {
        cdx[i] = std::max(-40000, std::min(40000, h_dx[i]));
        cdy[i] = std::max(-40000, std::min(40000, h_dy[i]));
    }
    const int n_rows = row_end - row_begin;
    const int tiles_x = (W + PR_TW - 1) / PR_TW, tiles_y = (n_rows + PR_TH - 1) / PR_TH;
    Planner pl;
    pl.T = T; pl.n_vel = n_vel; pl.ring_bytes = ring_bytes_for(T);
    pl.max_region = (pl.ring_bytes / 2 / 1024) * 1024;
    pl.dx = cdx.data(); pl.dy = cdy.data();
    int t_far = 0;
    {   // epoch with the largest displacement spread
        long long best = -1;
        for (int t = 0; t < T; ++t) {
            long long s = 0;
            for (int v = 0; v < n_vel; v += std::max(1, n_vel / 64)) s += llabs((long long)cdx[(size_t)v * T + t]) + llabs((long long)cdy[(size_t)v * T + t]);
            if (s > best) { best = s; t_far = t; }
        }
    }
    pl.idx.resize(n_vel); pl.px.resize(n_vel); pl.py.resize(n_vel);
    for (int v = 0; v < n_vel; ++v) {
        pl.idx[v] = v;
        pl.px[v] = cdx[(size_t)v * T + t_far];
        pl.py[v] = cdy[(size_t)v * T + t_far];
    }
    if (n_vel > 0) pl.split(0, n_vel);
    const int ng = (int)pl.leaves.size();
    // tables: gvel, per-group blocks {offs[T][G], ge[T]}, ring chain
    std::vector<int32_t>& gvel = PC.gvel;
    std::vector<unsigned char>& gtbl = PC.gtbl;
    gvel.assign((size_t)ng * PR_G, -1);
    gtbl.assign((size_t)ng * TBL, 0);
    double staged = 0.0, evals = 0.0, gathers = 0.0;
    uint32_t ph = 0;
    for (int g = 0; g < ng; ++g) {
        if (g % PR_SUB == 0) ph = 0;  // every work unit starts its ring chain at offset 0
        const int lo = pl.leaves[g].first, cnt = pl.leaves[g].second - pl.leaves[g].first;
        for (int j = 0; j < cnt; ++j) gvel[(size_t)g * PR_G + j] = pl.idx[lo + j];
        int32_t* offs = reinterpret_cast<int32_t*>(gtbl.data() + (size_t)g * TBL);
        GroupEpoch* ge = reinterpret_cast<GroupEpoch*>(gtbl.data() + (size_t)g * TBL + (size_t)T * PR_G * 4);
        for (int t = 0; t < T; ++t) {
            GroupEpoch e;
            memset(&e, 0, sizeof(e));
            int x0, y0;
            const long long bytes = pl.region(lo, lo + cnt, t, &e, &x0, &y0);
            KB_REQUIRE(bytes > 0 && bytes <= pl.max_region, KBMOD_ERR_UNSUPPORTED, "planner: region of %lld bytes", bytes);
            const int pitch = PR_TW + 16 * (int)(e.pitch_k & 0xFF);
            for (int j = 0; j < cnt; ++j) {
                const int v = pl.idx[lo + j];
                offs[t * PR_G + j] = ((cdy[(size_t)v * T + t] - y0) * pitch + (cdx[(size_t)v * T + t] - x0)) * (int)sizeof(unsigned int);
            }
            uint32_t pad = 0;
            if (ph + (uint32_t)bytes > (uint32_t)pl.ring_bytes) { pad = (uint32_t)pl.ring_bytes - ph; ph = 0; }
            e.smem_off = ph;
            e.footprint = (uint32_t)bytes + pad;
            e.vmask = cnt >= 32 ? 0xFFFFFFFFu : ((1u << cnt) - 1u);
            bool same = true;
            for (int j = 1; j < cnt; ++j) same = same && offs[t * PR_G + j] == offs[t * PR_G];
            if (same) e.pitch_k |= 0x100;
            gathers += (double)PR_TW * PR_TH * (same ? 1 : cnt);  // a uniform epoch is gathered once per pixel
            ph += (uint32_t)bytes;
            ge[t] = e;
            staged += (double)bytes;
        }
        evals += (double)PR_TW * PR_TH * cnt * T;
    }
    // on-image masks: region t of group g touches the image iff the tile column AND the tile row allow it
    // (tile row r of the band starts at image row row_begin + r * PR_TH)
    std::vector<unsigned long long>&maskx = PC.maskx, &masky = PC.masky;
    std::vector<uint32_t>& gfoot = PC.gfoot;
    maskx.assign((size_t)ng * tiles_x, 0ull);
    masky.assign((size_t)ng * tiles_y, 0ull);
    gfoot.assign((size_t)ng, 0u);
    double on = 0.0, all = 0.0;
    for (int g = 0; g < ng; ++g) {
        const GroupEpoch* ge = reinterpret_cast<const GroupEpoch*>(gtbl.data() + (size_t)g * TBL + (size_t)T * PR_G * 4);
        unsigned long long foot = 0;
        for (int t = 0; t < T; ++t) {
            const long long pitch = PR_TW + 16 * (long long)(ge[t].pitch_k & 0xFF), rows = (long long)ge[t].n_box * PR_RB;
            for (int c = 0; c < tiles_x; ++c) {
                const long long x0 = (long long)c * PR_TW + ge[t].ox;
                if (x0 < W && x0 + pitch > 0) maskx[(size_t)g * tiles_x + c] |= 1ull << t;
            }
            for (int r = 0; r < tiles_y; ++r) {
                const long long y0 = (long long)row_begin + (long long)r * PR_TH + ge[t].oy;
                if (y0 < H && y0 + rows > 0) masky[(size_t)g * tiles_y + r] |= 1ull << t;
            }
            foot += ge[t].footprint;
        }
        gfoot[g] = (uint32_t)std::min<unsigned long long>(foot, 0xFFFFFFFFull);  // > ring / 2 is all that matters
        for (int c = 0; c < tiles_x; ++c)
            for (int r = 0; r < tiles_y; ++r) {
                on += (double)__builtin_popcountll(maskx[(size_t)g * tiles_x + c] & masky[(size_t)g * tiles_y + r]);
                all += (double)T;
            }
    }
    PC.T = T; PC.H = H; PC.W = W; PC.row_begin = row_begin; PC.row_end = row_end; PC.n_vel = n_vel;
    PC.ng = ng; PC.staged = staged; PC.evals = evals;
    PC.gather_fraction = evals > 0 ? gathers / evals : 1.0;
    PC.off_image = all > 0 ? 1.0 - on / all : 0.0;
    PC.ring_bytes = ring_bytes_for(T);
    PC.tiles_x = tiles_x; PC.tiles_y = tiles_y;
    PC.too_scattered = (size_t)ng > max_groups(n_vel) ? 1 : 0;
    return KBMOD_OK;
}

// m(n): a lower bound on the number of epochs the sigma-G filter keeps out of n valid ones.  The clip window is
// [P50 - w, P50 + w], w = n_sigma C (P_hi - P_lo); with n_sigma C >= 1 (1e-3 of margin absorbs the float32
// roundings) and P_lo <= P50 <= P_hi it contains [P_lo, P_hi], hence every sample whose sorted index lies in
// [k_lo (+1 if P_lo is interpolated above s[k_lo]), k_hi].  Nearest rank: k = the rank itself, no interpolation.
static bool bound_min_kept(const kbmod_search_params* p, const DevParams& P, int T, BoundParams* bp) {
    const float prod = p->n_sigma * p->sigmag_coeff;
    for (int n = 0; n <= KBMOD_MAX_T; ++n) {
        int m = 1;
        if (n >= 1 && n <= T) {
            if (!P.sigmag_enable) m = n;
            else if (prod >= 1.001f && p->pct_lo <= 50.0f && p->pct_hi >= 50.0f) {
                // an interpolation weight within 1e-6 of 1 could round the interpolant onto (or past) s[k+1]: no claim
                const bool g_ok = P.fr_lo[n] < 1.0f - 1e-6f && P.fr_hi[n] < 1.0f - 1e-6f && P.fr_md[n] < 1.0f - 1e-6f;
                const int first = P.rk_lo[n] + (P.fr_lo[n] > 0.0f ? 1 : 0);
                m = g_ok ? std::max(1, (int)P.rk_hi[n] - first + 1) : 1;
            } else if (prod >= 0.0f && p->n_sigma >= 0.0f) m = 1;
            else return false;
        }
        bp->mkept[n] = (unsigned char)(n == 0 ? 0 : m);
    }
    {
        const int need = p->min_obs > 1 ? p->min_obs : 1;
        int mk = KBMOD_MAX_T;
        for (int n = need; n <= T; ++n) mk = std::min(mk, (int)bp->mkept[n]);
        bp->mk_min = need <= T ? mk : 0;
    }
    bp->pass_all = !(p->min_lh > 0.0f && p->min_lh < INFINITY);
    bp->cbits = 1;
    while ((1 << bp->cbits) <= T) ++bp->cbits;  // counts up to T fit: 2^cbits > T  (T = 26 -> 5, T = 64 -> 7)
    return true;
}

int kb_launch_search_pruned(const float* d_psiphi, const PrunedPlan& plan, const PrunedTablesDev& tbd, int TPv,
                            const void* d_S4, const S4Geom& G, const int* d_off, const kbmod_search_params* p,
                            const DevParams& P, unsigned long long* d_keys, void* d_scratch, size_t scratch_bytes,
                            unsigned long long* d_stats, cudaStream_t st, int* n_launches) {
    BoundParams bp;
    if (!bound_min_kept(p, P, plan.T, &bp)) {
        kb_set_error("pruned search needs n_sigma >= 0 and n_sigma*coeff >= 0");
        return KBMOD_ERR_UNSUPPORTED;
    }
    const int T = plan.T, H = plan.H, W = plan.W, n_vel = plan.n_vel, ng = plan.ng;
    const int row_begin = plan.row_begin, row_end = plan.row_end, n_rows = row_end - row_begin;
    const int TBL = tbl_bytes(T);
    const size_t ngm = max_groups(n_vel);
    KB_REQUIRE(!plan.too_scattered && (size_t)ng <= ngm, KBMOD_ERR_UNSUPPORTED,
               "pruned search: %d velocity groups needed, workspace holds %zu (velocities too scattered; use the direct kernel)",
               ng, ngm);
    // launches cover (a batch of whole waves of tiles) x (a chunk of the groups), sized so that 1/16 of the launch's
    // trajectories fit the survivor queue: 1.5 % survive on configs[2], 2.6 % on configs[3] (unevenly over the image);
    // what does not fit is evaluated wholesale by the overflow kernel (correct, 65 x the work for the items concerned).
    // Measured on configs[2] with a 2^28-entry queue for 1/4, 1/16, 1/24, 1/32, 1/64: bound phase 226.7 / 222.8 /
    // 218.4 / 221.1 / 217.0 ms (fewer launch tails, more L2 reuse of the staged planes), exact phase 82 ms except at
    // 1/64, where the queue overflows (169 ms); at 1/24 configs[3] overflowed on some launches.  Hence a larger queue
    // (2^29 entries) at 1/16, and batches of equal size (work units are handed out dynamically: whole waves do not matter).
    int n_sm = 148, dev = 0;
    KB_CUDA(cudaGetDevice(&dev));
    KB_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    const int n_tiles = (int)n_tiles_of(n_rows, W);
    const int grid = std::max(1, std::min(n_sm, n_tiles));
    const double budget = 16.0 * (double)queue_cap(n_vel);
    const double wave_nominal = (double)grid * PR_TW * PR_TH * (double)ng * PR_G;  // one wave, all groups
    const int n_chunks = std::max(1, std::min(std::max(ng, 1), (int)ceil(wave_nominal / budget)));
    const int groups_per_chunk = ((std::max(1, (ng + n_chunks - 1) / n_chunks) + PR_SUB - 1) / PR_SUB) * PR_SUB;

    // ---- scratch carve-up
    const ScratchLayout L = scratch_layout(T, H, W, n_rows, n_vel);
    KB_REQUIRE(L.total <= scratch_bytes, KBMOD_ERR_WORKSPACE, "pruned search scratch: need %zu, have %zu", L.total, scratch_bytes);
    const size_t Wp = ((size_t)W + 3) & ~(size_t)3;
    KB_REQUIRE((double)T * H * Wp < 2147483648.0, KBMOD_ERR_UNSUPPORTED, "T*H*Wp exceeds 2^31");
    char* w = (char*)d_scratch;
    unsigned int* d_B = (unsigned int*)(w + L.B);
    Queue Qu;
    Qu.entries = (uint2*)(w + L.qentries);
    Qu.count = (unsigned long long*)(w + L.qcount);
    Qu.units = Qu.count + 1;
    float* d_scale = (float*)(w + L.qcount + 256);  // unit, cap, floors and thresholds of the fixed-point bound planes
    unsigned int* d_thrtab = (unsigned int*)(w + L.qcount + 256 + al256(SC_FLOATS * sizeof(float)));
    Qu.cap = queue_cap(n_vel);
    Qu.overflow = (unsigned int*)(w + L.overflow);

    KB_CUDA(cudaMemsetAsync(d_keys, 0, (size_t)n_rows * W * P.K * 8, st));
    KB_CUDA(cudaMemsetAsync(Qu.overflow, 0, L.overflow_words * 4, st));

    // ---- tensor maps over the bound planes: uint32 elements, dims {Wp, H, T}
    kb_encode_tiled_fn enc = kb_get_encode_tiled();
    KB_REQUIRE(enc != nullptr, KBMOD_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
    TensorMaps maps;
    for (int hc = 0; hc < PR_NHEIGHT; ++hc)
        for (int k = 0; k < PR_NPITCH; ++k) {
            cuuint64_t dims[3] = {(cuuint64_t)Wp, (cuuint64_t)H, (cuuint64_t)T};
            cuuint64_t strides[2] = {(cuuint64_t)Wp * 4, (cuuint64_t)Wp * 4 * (cuuint64_t)H};
            cuuint32_t box[3] = {(cuuint32_t)(PR_TW + 16 * k), (cuuint32_t)(PR_RB << hc), 1};
            cuuint32_t estr[3] = {1, 1, 1};
            CUresult r = enc(&maps.m[hc * PR_NPITCH + k], CU_TENSOR_MAP_DATA_TYPE_UINT32, 3, (void*)d_B, dims, strides, box, estr,
                             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            KB_REQUIRE(r == CUDA_SUCCESS, KBMOD_ERR_CUDA, "cuTensorMapEncodeTiled failed with %d (pitch %d, %d rows)", (int)r,
                       PR_TW + 16 * k, PR_RB << hc);
        }

    // ---- launches
    int launches = 0;
    {
        const size_t n = (size_t)T * H * Wp;
        bound_scale_kernel<<<1, 1024, 0, st>>>(reinterpret_cast<const float2*>(d_psiphi), T, H, W, P.min_lh, bp,
                                               P.min_obs > 1 ? P.min_obs : 1, d_scale, d_thrtab);
        KB_CUDA(cudaGetLastError());
        bound_plane_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(reinterpret_cast<const float2*>(d_psiphi), d_B, H, W,
                                                                        (int)Wp, (size_t)T * H, bp.cbits, d_scale);
        KB_CUDA(cudaGetLastError());
        launches += 2;
        kb_phase_mark(KB_PHASE_PLANES, st);
    }
    const double tile_nominal = (double)PR_TW * PR_TH * (double)groups_per_chunk * PR_G;  // one tile, one chunk of groups
    long long per_launch = (long long)(budget / std::max(1.0, tile_nominal));
    per_launch = std::max<long long>(grid, std::min<long long>((long long)PR_WAVES_PER_BATCH * grid, per_launch));
    const long long n_batches = ((long long)n_tiles + per_launch - 1) / per_launch;
    const int batch = (int)(((long long)n_tiles + n_batches - 1) / n_batches);
    const size_t smem1 = (size_t)plan.ring_bytes + (size_t)PR_NTBL * TBL + PR_SMEM_MISC;
    KB_CUDA(cudaFuncSetAttribute(bound_phase_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem1));
    PrunedTables tb{tbd.gvel, tbd.gtbl, tbd.maskx, tbd.masky, tbd.gfoot, ng, plan.ring_bytes};
    ExactArgs EA{reinterpret_cast<const float2*>(d_S4), G, d_off, W, row_begin, row_end, d_keys};
    KB_DISPATCH_TP(TPv, {
        const size_t smem2 = (size_t)TP * EX_THREADS * sizeof(float);
        const size_t smem2q = (size_t)TP * ExCfg<TP>::threads * sizeof(float);
        KB_CUDA(cudaFuncSetAttribute(exact_queue_kernel<TP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2q));
        KB_CUDA(cudaFuncSetAttribute(exact_overflow_kernel<TP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
        if (ng > 0) {
            for (int b0 = 0; b0 < n_tiles; b0 += batch) {
                const int b1 = std::min(n_tiles, b0 + batch);
                for (int g0 = 0; g0 < ng; g0 += groups_per_chunk) {
                    const int g1 = std::min(ng, g0 + groups_per_chunk);
                    KB_CUDA(cudaMemsetAsync(Qu.count, 0, 3 * sizeof(unsigned long long), st));  // queue, unit and chunk counters
                    bound_phase_kernel<<<std::min(grid, b1 - b0), PR_THREADS, smem1, st>>>(maps, T, row_begin, row_end, W, b0, b1,
                                                                                          g0, g1, tb, bp, P.min_obs, d_thrtab, Qu);
                    KB_CUDA(cudaGetLastError());
                    kb_phase_mark(KB_PHASE_BOUND, st);
                    exact_queue_kernel<TP><<<n_sm * ExCfg<TP>::ctas, ExCfg<TP>::threads, smem2q, st>>>(EA, P, Qu, d_stats);
                    KB_CUDA(cudaGetLastError());
                    kb_phase_mark(KB_PHASE_EXACT, st);
                    launches += 2;
                }
            }
            exact_overflow_kernel<TP><<<n_sm * EX_CTAS_PER_SM, EX_THREADS, smem2, st>>>(EA, P, Qu.overflow, L.overflow_words,
                                                                                       tbd.gvel, ng, d_stats);
            kb_phase_mark(KB_PHASE_EXACT, st);
            ++launches;
        }
    });
    KB_CUDA(cudaGetLastError());
    if (n_launches) *n_launches = launches;
    return KBMOD_OK;
}
