// Measurement helper for the roofline denominator ("re-measure the SMEM peak with an LDS microbenchmark
// at the clocks the kernel actually holds"): every SM streams conflict-free shared-memory loads of 4, 8 or 16 bytes
// per lane, many independent loads in flight per thread, nothing else in the loop.  Not part of the search path.
#include "common.cuh"

namespace {

constexpr int SP_THREADS = 1024, SP_LOADS = 8;  // 8 distinct vectors per thread and iteration: 8 x 1024 x sizeof(V) bytes

template <typename V>
__global__ void __launch_bounds__(SP_THREADS) smem_peak_kernel(int iters, unsigned int* __restrict__ sink) {
    extern __shared__ __align__(16) unsigned int buf[];
    constexpr int PER = sizeof(V) / 4;                  // words per lane and load
    constexpr int NV = SP_LOADS * SP_THREADS;           // vectors in the buffer
    for (int i = threadIdx.x; i < NV * PER; i += SP_THREADS) buf[i] = i * 2654435761u;
    __syncthreads();
    const V* v = reinterpret_cast<const V*>(buf);
    unsigned int acc = 0;
    int idx = threadIdx.x;                              // consecutive lanes -> consecutive vectors: conflict-free
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < SP_LOADS; ++u) {
            const V x = v[(idx + u * SP_THREADS) & (NV - 1)];
            const unsigned int* w = reinterpret_cast<const unsigned int*>(&x);
#pragma unroll
            for (int k = 0; k < PER; ++k) acc += w[k];
        }
        idx = (idx + 32) & (NV - 1);                    // another warp's vectors next time: nothing to hoist
    }
    if (acc == 0x12345678u) sink[0] = acc;              // keeps the loads alive
}

template <typename V>
int run_peak(int iters, int grid, unsigned int* sink, cudaStream_t st) {
    const int smem = SP_LOADS * SP_THREADS * (int)sizeof(V);
    KB_CUDA(cudaFuncSetAttribute(smem_peak_kernel<V>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    smem_peak_kernel<V><<<grid, SP_THREADS, smem, st>>>(iters, sink);
    return KBMOD_OK;
}

}  // namespace

extern "C" int kbmod_measure_smem_gbs(int bytes_per_lane, void* d_scratch4, double* h_gbs, void* stream) {
    KB_REQUIRE(h_gbs && d_scratch4, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(bytes_per_lane == 4 || bytes_per_lane == 8 || bytes_per_lane == 16, KBMOD_ERR_INVALID_ARG,
               "bytes_per_lane = %d must be 4, 8 or 16", bytes_per_lane);
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, n_sm = 0;
    KB_CUDA(cudaGetDevice(&dev));
    KB_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    unsigned int* sink = (unsigned int*)d_scratch4;  // caller-owned: the library never allocates device memory
    cudaEvent_t e0, e1;
    KB_CUDA(cudaEventCreate(&e0));
    KB_CUDA(cudaEventCreate(&e1));
    const int iters = 8000, grid = n_sm;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {  // first repetition warms up
        KB_CUDA(cudaEventRecord(e0, st));
        int rc = bytes_per_lane == 4 ? run_peak<unsigned int>(iters, grid, sink, st)
                 : bytes_per_lane == 8 ? run_peak<uint2>(iters, grid, sink, st) : run_peak<uint4>(iters, grid, sink, st);
        if (rc) return rc;
        KB_CUDA(cudaEventRecord(e1, st));
        KB_CUDA(cudaEventSynchronize(e1));
        float ms = 0.0f;
        KB_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        const double bytes = (double)grid * SP_THREADS * (double)iters * SP_LOADS * bytes_per_lane;
        if (rep > 0) best = fmax(best, bytes / (ms * 1e-3) / 1e9);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    KB_CUDA(cudaGetLastError());
    *h_gbs = best;
    return KBMOD_OK;
}

// ---------------------------------------------------------------------------------------------
// Issue rate of a few opcodes (warp-instructions per clock per SM), measured the same way: 8 independent chains per
// thread, 32 warps per SM, nothing else in the loop.  What it is for: on sm_100a FMNMX (like LOP3, IMAD, IMNMX) issues
// on the half-rate ALU pipe, IADD3 (two register operands) and FADD at the full rate.  An exchange built from one FMNMX
// and a three-register IADD3 (maximum = a + b - min on the bit patterns) was tried for that reason and runs at 0.83
// exchanges per clock per SM against 0.99 for two FMNMX: op 3 keeps the measurement.
namespace {

constexpr int IR_CHAINS = 8, IR_ITERS = 4096;

template <int OP>
__global__ void __launch_bounds__(1024) issue_rate_kernel(int iters, float a0, unsigned int* __restrict__ sink) {
    float x[IR_CHAINS], y[IR_CHAINS];
    int ix[IR_CHAINS];
#pragma unroll
    for (int i = 0; i < IR_CHAINS; ++i) {
        x[i] = a0 + threadIdx.x * 1e-3f + i;
        y[i] = 2.0f * a0 - i;
        ix[i] = threadIdx.x + i;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < IR_CHAINS; ++i) {
            if (OP == 0) {  // two FMNMX (min, max on different chains so that ptxas cannot fuse them into FMNMX3)
                asm volatile("min.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(y[(i + 1) % IR_CHAINS]));
                asm volatile("max.f32 %0, %0, %1;" : "+f"(y[i]) : "f"(x[(i + 3) % IR_CHAINS]));
            }
            if (OP == 1) {  // two integer adds
                asm volatile("add.s32 %0, %0, %1;" : "+r"(ix[i]) : "r"(ix[(i + 1) % IR_CHAINS]));
                asm volatile("add.s32 %0, %0, %1;" : "+r"(ix[(i + 2) % IR_CHAINS]) : "r"(it));
            }
            if (OP == 2) {  // two FADD
                asm volatile("add.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(y[(i + 1) % IR_CHAINS]));
                asm volatile("add.f32 %0, %0, %1;" : "+f"(y[i]) : "f"(x[(i + 3) % IR_CHAINS]));
            }
            if (OP == 3) {  // the alternative compare-exchange: FMNMX + (a + b - min) on the bit patterns
                const float lo = fminf(x[i], y[i]);
                y[i] = __int_as_float(__float_as_int(x[i]) + __float_as_int(y[i]) - __float_as_int(lo));
                x[i] = lo + a0;  // keeps the chain alive (one FADD)
            }
        }
    }
    float s = 0.0f;
    int si = 0;
#pragma unroll
    for (int i = 0; i < IR_CHAINS; ++i) {
        s += x[i] + y[i];
        si += ix[i];
    }
    if (s + (float)si == a0 * 7.25f) sink[0] = (unsigned int)si;
}

}  // namespace

// op: 0 = FMNMX, 1 = IADD3, 2 = FADD, 3 = the alternative compare-exchange (FMNMX + three-register IADD3 + FADD).  *h_rate = warp-instructions of the
// loop body per SM clock (max SM clock) per SM: 2 per chain step for op 0-2, 3 for op 3.
extern "C" int kbmod_measure_issue_rate(int op, void* d_scratch4, double* h_rate, void* stream) {
    KB_REQUIRE(h_rate && d_scratch4, KBMOD_ERR_INVALID_ARG, "NULL argument");
    KB_REQUIRE(op >= 0 && op <= 3, KBMOD_ERR_INVALID_ARG, "op = %d must be 0..3", op);
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, n_sm = 0, khz = 0;
    KB_CUDA(cudaGetDevice(&dev));
    KB_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    KB_CUDA(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
    cudaEvent_t e0, e1;
    KB_CUDA(cudaEventCreate(&e0));
    KB_CUDA(cudaEventCreate(&e1));
    unsigned int* sink = (unsigned int*)d_scratch4;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        KB_CUDA(cudaEventRecord(e0, st));
        if (op == 0) issue_rate_kernel<0><<<n_sm * 2, 1024, 0, st>>>(IR_ITERS, 1.0f, sink);
        if (op == 1) issue_rate_kernel<1><<<n_sm * 2, 1024, 0, st>>>(IR_ITERS, 1.0f, sink);
        if (op == 2) issue_rate_kernel<2><<<n_sm * 2, 1024, 0, st>>>(IR_ITERS, 1.0f, sink);
        if (op == 3) issue_rate_kernel<3><<<n_sm * 2, 1024, 0, st>>>(IR_ITERS, 1.0f, sink);
        KB_CUDA(cudaEventRecord(e1, st));
        KB_CUDA(cudaEventSynchronize(e1));
        float ms = 0.0f;
        KB_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        const double winst = (double)n_sm * 2 * 32 * (double)IR_ITERS * IR_CHAINS * (op == 3 ? 3 : 2);
        const double clk = (double)ms * 1e-3 * (double)khz * 1e3;
        if (rep > 0) best = fmax(best, winst / clk / n_sm);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    KB_CUDA(cudaGetLastError());
    *h_rate = best;
    return KBMOD_OK;
}
