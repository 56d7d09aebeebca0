// (a1) psi/phi preparation -- PAPER.md:L79 (s3), readings R1-R4 (see include/kbmod_b200.h).
//   Psi = P (*) (I w),  Phi = P^2 (*) w,  w = 1/var on good pixels and 0 elsewhere (correlation).
// One launch per epoch; the epoch's PSF travels in the kernel parameter bank (<= 31*31 floats).
//
// Kernel shape: a block computes a PREP_TX x PREP_TY tile of outputs.  The (I w, w) pairs of the
// tile plus its PSF halo are staged once in shared memory (coalesced reads of img / var / mask:
// 9 B per pixel, the algorithmic minimum, plus the halo overlap), then every thread produces
// PREP_R vertically adjacent outputs, sliding a register window down each kernel column so that
// one shared-memory read feeds up to PREP_R multiply-adds per plane.
#include <math.h>

#include "common.cuh"

namespace {

constexpr int PREP_TX = 32;          // outputs per block in x  (one warp-row)
constexpr int PREP_R = 8;            // outputs per thread in y
constexpr int PREP_WARPS = 8;        // warps per block
constexpr int PREP_TY = PREP_R * PREP_WARPS;

struct PsfParam {
    float p[KBMOD_MAX_PSF * KBMOD_MAX_PSF];
};

template <int KS>  // KS = compile-time PSF side, or 0 for a run-time side
__global__ void __launch_bounds__(PREP_TX* PREP_WARPS)
prep_kernel(const float* __restrict__ img, const float* __restrict__ var, const uint8_t* __restrict__ mask, int H,
            int W, int k_rt, const __grid_constant__ PsfParam psf, float2* __restrict__ out) {
    const int k = KS ? KS : k_rt;
    const int r = k / 2;
    extern __shared__ float2 tile[];  // [(PREP_TY + k - 1)][pitch]
    const int pitch = PREP_TX + k - 1;
    const int rows = PREP_TY + k - 1;
    const int x_org = blockIdx.x * PREP_TX - r;
    const int y_org = blockIdx.y * PREP_TY - r;
    const int tid = threadIdx.y * PREP_TX + threadIdx.x;

    for (int idx = tid; idx < rows * pitch; idx += PREP_TX * PREP_WARPS) {
        const int ty = idx / pitch, tx = idx - ty * pitch;
        const int x = x_org + tx, y = y_org + ty;
        float2 v = make_float2(0.0f, 0.0f);
        if (x >= 0 && x < W && y >= 0 && y < H) {
            const size_t q = (size_t)y * W + x;
            const float I = __ldg(img + q), V = __ldg(var + q);
            const bool bad = (mask && __ldg(mask + q) != 0) || !(V > 0.0f) || !isfinite(V) || !isfinite(I);
            if (!bad) {
                const float w = 1.0f / V;
                v = make_float2(I * w, w);
            }
        }
        tile[idx] = v;
    }
    __syncthreads();

    float ps[PREP_R], ph[PREP_R];
#pragma unroll
    for (int a = 0; a < PREP_R; ++a) ps[a] = ph[a] = 0.0f;
    const int ly = threadIdx.y * PREP_R;  // first output row of this thread inside the tile
    const int lx = threadIdx.x;

    // out(ly+a) = sum_j sum_i P[j][i] * tile[ly+a+j][lx+i].  For a fixed column i walk jj = a + j
    // down the column: each value read once, used by every output row a with 0 <= jj-a < k.
#pragma unroll 1
    for (int i = 0; i < k; ++i) {
        const float2* col = tile + (size_t)ly * pitch + lx + i;
#pragma unroll 1
        for (int jj = 0; jj < k + PREP_R - 1; ++jj) {
            const float2 v = col[jj * pitch];
#pragma unroll
            for (int a = 0; a < PREP_R; ++a) {
                const int j = jj - a;
                if (j >= 0 && j < k) {
                    const float p = psf.p[j * k + i];
                    ps[a] = fmaf(p, v.x, ps[a]);
                    ph[a] = fmaf(p * p, v.y, ph[a]);
                }
            }
        }
    }

    const int x = blockIdx.x * PREP_TX + lx;
    if (x < W) {
#pragma unroll
        for (int a = 0; a < PREP_R; ++a) {
            const int y = blockIdx.y * PREP_TY + ly + a;
            if (y < H) {
                const float wc = tile[(size_t)(ly + a + r) * pitch + lx + r].y;
                out[(size_t)y * W + x] = (wc > 0.0f) ? make_float2(ps[a], ph[a]) : make_float2(0.0f, 0.0f);
            }
        }
    }
}

// Separable PSFs (P[j][i] = u[j] v[i], e.g. any Gaussian): a row pass into a second shared-memory array, then a
// column pass with the same sliding register window: k + k (1 + (k-1)/64) multiply-adds per plane and output
// instead of k^2 (29 instead of 169 for the 13x13 PSF of the DECam-shaped configs).
struct SepParam {
    float u[KBMOD_MAX_PSF], v[KBMOD_MAX_PSF];    // column (y) and row (x) factors
    float u2[KBMOD_MAX_PSF], v2[KBMOD_MAX_PSF];  // their float32 squares (the weights of the phi plane)
};

// The same two passes with the PSF side as a template parameter: every loop over taps is unrolled, the taps are
// immediate operands from the parameter bank, the squares come precomputed, staging walks (row, x) without a
// division.  64 x 64 outputs per block of 512 threads (1.41 x halo for a 13 x 13 PSF instead of 1.63 x), two blocks
// per SM.  Same order of multiply-adds as prep_sep_kernel: the results are the same bits.
constexpr int PS_TX = 64, PS_TY = 64, PS_THREADS = 512, PS_WARPS = PS_THREADS / 32, PS_R = 8;
static_assert(PS_TX * (PS_TY / PS_R) == PS_THREADS, "column pass: one thread per (x, group of PS_R rows)");

template <int K>
__global__ void __launch_bounds__(PS_THREADS, 2)
prep_sep_kernel_k(const float* __restrict__ img, const float* __restrict__ var, const uint8_t* __restrict__ mask, int H,
                  int W, const __grid_constant__ SepParam psf, float2* __restrict__ out) {
    constexpr int R = K / 2, PITCH = PS_TX + K - 1, ROWS = PS_TY + K - 1;
    extern __shared__ float2 tile[];  // [ROWS][PITCH], then the row-pass result [ROWS][PS_TX]
    float2* hp = tile + ROWS * PITCH;
    const int x_org = blockIdx.x * PS_TX - R, y_org = blockIdx.y * PS_TY - R;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int ty = warp; ty < ROWS; ty += PS_WARPS) {
        const int y = y_org + ty;
        const bool y_in = y >= 0 && y < H;
        for (int tx = lane; tx < PITCH; tx += 32) {
            const int x = x_org + tx;
            float2 v = make_float2(0.0f, 0.0f);
            if (y_in && x >= 0 && x < W) {
                const size_t q = (size_t)y * W + x;
                const float I = __ldg(img + q), V = __ldg(var + q);
                const bool bad = (mask && __ldg(mask + q) != 0) || !(V > 0.0f) || !isfinite(V) || !isfinite(I);
                if (!bad) {
                    const float w = 1.0f / V;
                    v = make_float2(I * w, w);
                }
            }
            tile[ty * PITCH + tx] = v;
        }
    }
    __syncthreads();
    // row pass: hp[row][x] = sum_i v[i] tile[row][x + i]  (v[i]^2 for the weight plane)
    for (int row = warp; row < ROWS; row += PS_WARPS) {
#pragma unroll
        for (int c = 0; c < PS_TX / 32; ++c) {
            const float2* src = tile + row * PITCH + c * 32 + lane;
            float a = 0.0f, b = 0.0f;
#pragma unroll
            for (int i = 0; i < K; ++i) {
                const float2 t = src[i];
                a = fmaf(psf.v[i], t.x, a);
                b = fmaf(psf.v2[i], t.y, b);
            }
            hp[row * PS_TX + c * 32 + lane] = make_float2(a, b);
        }
    }
    __syncthreads();
    // column pass: out(ly + a) = sum_j u[j] hp[ly + a + j], a register window sliding down the column
    const int lx = threadIdx.x % PS_TX, ly = (threadIdx.x / PS_TX) * PS_R;
    float ps[PS_R], ph[PS_R];
#pragma unroll
    for (int a = 0; a < PS_R; ++a) ps[a] = ph[a] = 0.0f;
    const float2* col = hp + ly * PS_TX + lx;
#pragma unroll
    for (int jj = 0; jj < K + PS_R - 1; ++jj) {
        const float2 t = col[jj * PS_TX];
#pragma unroll
        for (int a = 0; a < PS_R; ++a) {
            const int j = jj - a;
            if (j >= 0 && j < K) {
                ps[a] = fmaf(psf.u[j], t.x, ps[a]);
                ph[a] = fmaf(psf.u2[j], t.y, ph[a]);
            }
        }
    }
    const int x = blockIdx.x * PS_TX + lx;
    if (x < W) {
#pragma unroll
        for (int a = 0; a < PS_R; ++a) {
            const int y = blockIdx.y * PS_TY + ly + a;
            if (y < H) {
                const float wc = tile[(ly + a + R) * PITCH + lx + R].y;
                out[(size_t)y * W + x] = (wc > 0.0f) ? make_float2(ps[a], ph[a]) : make_float2(0.0f, 0.0f);
            }
        }
    }
}

template <int K>
static int launch_sep_k(const float* img, const float* var, const uint8_t* mask, int H, int W, const SepParam& sep,
                        float2* out, cudaStream_t st) {
    constexpr size_t smem = ((size_t)(PS_TY + K - 1) * (PS_TX + K - 1) + (size_t)(PS_TY + K - 1) * PS_TX) * sizeof(float2);
    KB_CUDA(cudaFuncSetAttribute(prep_sep_kernel_k<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const dim3 grid((W + PS_TX - 1) / PS_TX, (H + PS_TY - 1) / PS_TY);
    prep_sep_kernel_k<K><<<grid, PS_THREADS, smem, st>>>(img, var, mask, H, W, sep, out);
    return KBMOD_OK;
}

__global__ void __launch_bounds__(PREP_TX* PREP_WARPS)
prep_sep_kernel(const float* __restrict__ img, const float* __restrict__ var, const uint8_t* __restrict__ mask, int H,
                int W, int k, const __grid_constant__ SepParam psf, float2* __restrict__ out) {
    const int r = k / 2;
    extern __shared__ float2 tile[];  // [(PREP_TY + k - 1)][pitch], then the row-pass result [(PREP_TY + k - 1)][PREP_TX]
    const int pitch = PREP_TX + k - 1;
    const int rows = PREP_TY + k - 1;
    float2* hp = tile + rows * pitch;
    const int x_org = blockIdx.x * PREP_TX - r;
    const int y_org = blockIdx.y * PREP_TY - r;
    const int tid = threadIdx.y * PREP_TX + threadIdx.x;

    for (int idx = tid; idx < rows * pitch; idx += PREP_TX * PREP_WARPS) {
        const int ty = idx / pitch, tx = idx - ty * pitch;
        const int x = x_org + tx, y = y_org + ty;
        float2 v = make_float2(0.0f, 0.0f);
        if (x >= 0 && x < W && y >= 0 && y < H) {
            const size_t q = (size_t)y * W + x;
            const float I = __ldg(img + q), V = __ldg(var + q);
            const bool bad = (mask && __ldg(mask + q) != 0) || !(V > 0.0f) || !isfinite(V) || !isfinite(I);
            if (!bad) {
                const float w = 1.0f / V;
                v = make_float2(I * w, w);
            }
        }
        tile[idx] = v;
    }
    __syncthreads();
    // row pass: hp[row][x] = sum_i v[i] tile[row][x + i]  (and v[i]^2 for the weight plane)
    const int lx = threadIdx.x;
    for (int row = threadIdx.y; row < rows; row += PREP_WARPS) {
        const float2* src = tile + (size_t)row * pitch + lx;
        float a = 0.0f, b = 0.0f;
#pragma unroll 1
        for (int i = 0; i < k; ++i) {
            const float2 t = src[i];
            const float vi = psf.v[i];
            a = fmaf(vi, t.x, a);
            b = fmaf(vi * vi, t.y, b);
        }
        hp[row * PREP_TX + lx] = make_float2(a, b);
    }
    __syncthreads();
    // column pass: out(ly + a) = sum_j u[j] hp[ly + a + j]
    float ps[PREP_R], ph[PREP_R];
#pragma unroll
    for (int a = 0; a < PREP_R; ++a) ps[a] = ph[a] = 0.0f;
    const int ly = threadIdx.y * PREP_R;
    const float2* col = hp + (size_t)ly * PREP_TX + lx;
#pragma unroll 1
    for (int jj = 0; jj < k + PREP_R - 1; ++jj) {
        const float2 t = col[jj * PREP_TX];
#pragma unroll
        for (int a = 0; a < PREP_R; ++a) {
            const int j = jj - a;
            if (j >= 0 && j < k) {
                const float uj = psf.u[j];
                ps[a] = fmaf(uj, t.x, ps[a]);
                ph[a] = fmaf(uj * uj, t.y, ph[a]);
            }
        }
    }
    const int x = blockIdx.x * PREP_TX + lx;
    if (x < W) {
#pragma unroll
        for (int a = 0; a < PREP_R; ++a) {
            const int y = blockIdx.y * PREP_TY + ly + a;
            if (y < H) {
                const float wc = tile[(size_t)(ly + a + r) * pitch + lx + r].y;
                out[(size_t)y * W + x] = (wc > 0.0f) ? make_float2(ps[a], ph[a]) : make_float2(0.0f, 0.0f);
            }
        }
    }
}

// P = u v^T to float32 precision per tap?  (u[j] = P[j][c] / P[c][c], v[i] = P[c][i], c = k/2)
static bool separable(const float* P, int k, SepParam* sp) {
    const int c = k / 2;
    const double pc = (double)P[c * k + c];
    if (!(fabs(pc) > 0.0)) return false;
    double pmax = 0.0;
    for (int i = 0; i < k * k; ++i) pmax = fmax(pmax, fabs((double)P[i]));
    for (int j = 0; j < k; ++j)
        for (int i = 0; i < k; ++i) {
            const double want = (double)P[j * k + i], got = (double)P[j * k + c] / pc * (double)P[c * k + i];
            if (!(fabs(want - got) <= 2e-7 * fabs(want) + 1e-12 * pmax)) return false;
        }
    for (int j = 0; j < KBMOD_MAX_PSF; ++j) {
        sp->u[j] = j < k ? (float)((double)P[j * k + c] / pc) : 0.0f;
        sp->v[j] = j < k ? P[c * k + j] : 0.0f;
        sp->u2[j] = sp->u[j] * sp->u[j];  // float32 products, as the generic kernel forms them on the device
        sp->v2[j] = sp->v[j] * sp->v[j];
    }
    return true;
}

}  // namespace

int kb_launch_prep(const float* d_img, const float* d_var, const uint8_t* d_mask, int T, int H, int W,
                   const float* h_psf, int n_psf, int k, float* d_psiphi, cudaStream_t st) {
    const dim3 block(PREP_TX, PREP_WARPS);
    const dim3 grid((W + PREP_TX - 1) / PREP_TX, (H + PREP_TY - 1) / PREP_TY);
    const size_t smem = (size_t)(PREP_TY + k - 1) * (PREP_TX + k - 1) * sizeof(float2);
    const size_t plane = (size_t)H * W;
    PsfParam psf;
    SepParam sep;
    const size_t smem_sep = smem + (size_t)(PREP_TY + k - 1) * PREP_TX * sizeof(float2);
    KB_CUDA(cudaFuncSetAttribute(prep_sep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_sep));
    for (int t = 0; t < T; ++t) {
        const float* src = h_psf + (n_psf > 1 ? (size_t)t * k * k : 0);
        if (k > 1 && separable(src, k, &sep)) {
            const float* im = d_img + t * plane;
            const float* va = d_var + t * plane;
            const uint8_t* ma = d_mask ? d_mask + t * plane : nullptr;
            float2* o = reinterpret_cast<float2*>(d_psiphi) + t * plane;
            int rc = KBMOD_OK;
            bool instantiated = true;
            switch (k) {
#define KB_SEP_CASE(K) case K: rc = launch_sep_k<K>(im, va, ma, H, W, sep, o, st); break;
                KB_SEP_CASE(3) KB_SEP_CASE(5) KB_SEP_CASE(7) KB_SEP_CASE(9) KB_SEP_CASE(11) KB_SEP_CASE(13)
                KB_SEP_CASE(15) KB_SEP_CASE(17) KB_SEP_CASE(19) KB_SEP_CASE(21) KB_SEP_CASE(23) KB_SEP_CASE(25)
                KB_SEP_CASE(27) KB_SEP_CASE(29) KB_SEP_CASE(31)
#undef KB_SEP_CASE
                default: instantiated = false; break;
            }
            if (rc) return rc;
            if (instantiated) continue;
            prep_sep_kernel<<<grid, block, smem_sep, st>>>(d_img + t * plane, d_var + t * plane,
                                                           d_mask ? d_mask + t * plane : nullptr, H, W, k, sep,
                                                           reinterpret_cast<float2*>(d_psiphi) + t * plane);
            continue;
        }
        for (int i = 0; i < k * k; ++i) psf.p[i] = src[i];
        for (int i = k * k; i < KBMOD_MAX_PSF * KBMOD_MAX_PSF; ++i) psf.p[i] = 0.0f;
        prep_kernel<0><<<grid, block, smem, st>>>(d_img + t * plane, d_var + t * plane,
                                                  d_mask ? d_mask + t * plane : nullptr, H, W, k, psf,
                                                  reinterpret_cast<float2*>(d_psiphi) + t * plane);
    }
    KB_CUDA(cudaGetLastError());
    return KBMOD_OK;
}
