// k_probe.cu - MEASUREMENT UTILITIES, not part of the gridding path (SURVEY.md section 8(b) lists no such call): the
// denominators that bench.py and profiles/ compare the kernels against - FP32 FMA throughput (the second roofline term
// of BASELINE.json north_star) and the conflict-free shared-memory atomic rate (north_star: "shared-memory atomic
// throughput against the chip's peaks").
#include "plan.h"

// ---------------------------------------------------------------- FP32 peak probe (bench.py roofline denominator)
// Register-only dependent-chain-free FMA loops: 8 independent accumulators per thread, 4 resident CTAs of 256 threads
// per SM.  Variant 0 issues fma.rn.f32 (FFMA), variant 1 fma.rn.f32x2 (FFMA2, two fp32 FMAs per lane per instruction).
namespace mwa {

template <int VARIANT>
__global__ void __launch_bounds__(256) fp32_probe_kernel(float* out, int iters, float seed) {
    float a[8], b[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) { a[k] = seed + k + threadIdx.x; b[k] = seed * 0.5f + k; }
    const float m = 1.0000001f, c = 1e-7f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            if (VARIANT == 0) {
#pragma unroll
                for (int k = 0; k < 8; ++k) { a[k] = fmaf(a[k], m, c); b[k] = fmaf(b[k], m, c); }
            } else {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    unsigned long long v, mm, cc;
                    asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(a[k]), "f"(b[k]));
                    asm("mov.b64 %0, {%1, %1};" : "=l"(mm) : "f"(m));
                    asm("mov.b64 %0, {%1, %1};" : "=l"(cc) : "f"(c));
                    asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(v) : "l"(mm), "l"(cc));
                    asm("mov.b64 {%0, %1}, %2;" : "=f"(a[k]), "=f"(b[k]) : "l"(v));
                }
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k] + b[k];
    if (s == 12345.678f) out[0] = s;                               // keeps the loop alive
}

// Returns TFLOP/s (2 flop per FMA) of the two variants; synchronous on `st`.
bool probe_fp32(Plan* p, double* tflops_ffma, double* tflops_ffma2, cudaStream_t st) {
    float* d = nullptr;
    if (!cuda_ok(cudaMalloc((void**)&d, 4), "probe malloc")) return false;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 4096, blocks = p->sm_count * 8;
    double res[2] = {0, 0};
    for (int v = 0; v < 2; ++v) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {
            cudaEventRecord(e0, st);
            if (v == 0) fp32_probe_kernel<0><<<blocks, 256, 0, st>>>(d, iters, 1.0f);
            else fp32_probe_kernel<1><<<blocks, 256, 0, st>>>(d, iters, 1.0f);
            cudaEventRecord(e1, st);
            cudaEventSynchronize(e1);
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        const double fmas = (double)blocks * 256 * iters * 8 * 16;      // 16 fp32 FMAs per inner k-loop pass, 8 passes
        res[v] = 2.0 * fmas / (best * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    *tflops_ffma = res[0];
    *tflops_ffma2 = res[1];
    return cuda_ok(cudaGetLastError(), "fp32 probe");
}

// Conflict-free red.shared.add.f32: every lane of a warp adds to its own bank, 8 independent addresses per thread.
__global__ void __launch_bounds__(256) smem_atomic_probe_kernel(float* out, int iters) {
    __shared__ float cell[8 * 256];
    for (int k = threadIdx.x; k < 8 * 256; k += 256) cell[k] = 0.0f;
    __syncthreads();
    const unsigned a0 = (unsigned)__cvta_generic_to_shared(cell) + 4u * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) asm volatile("red.shared.add.f32 [%0], %1;" ::"r"(a0 + 1024u * k), "f"(1.0f) : "memory");
    }
    __syncthreads();
    if (cell[threadIdx.x] == 12345.678f) out[0] = cell[threadIdx.x];
}

// Lane-atomics per second over the whole device (divide by SMs x clock for the per-SM-per-clock figure).
bool probe_smem_atomics(Plan* p, double* lane_atomics_per_s, cudaStream_t st) {
    float* d = nullptr;
    if (!cuda_ok(cudaMalloc((void**)&d, 4), "probe malloc")) return false;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 2048, blocks = p->sm_count * 8;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        smem_atomic_probe_kernel<<<blocks, 256, 0, st>>>(d, iters);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    *lane_atomics_per_s = (double)blocks * 256 * iters * 8 / (best * 1e-3);
    return cuda_ok(cudaGetLastError(), "shared atomic probe");
}

}  // namespace mwa
