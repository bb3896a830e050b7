// bench_peak.cu -- register-only pipe-peak microbenchmarks for bench.py: the MEASURED denominators that ride beside the
// derived ALU roofline.  MEASURED_PEAKS.json only carries HBM and BF16 tensor numbers; the FMA-pipe
// kernels are bound by the FMA / FP64 / XU pipes, so those are measured here with the same clocks the kernels see.
// Bench-only helper: built into libbench_peak.so by bench.py / __graft_entry__.build(); NOT part of liblsp_b200.so or its ABI.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

namespace {

constexpr int kPeakThreads = 256;
constexpr int kPeakIters = 4096;
constexpr int kPeakIlp = 8;

// which = 0: FFMA (1 op / lane / instr)
__global__ void __launch_bounds__(kPeakThreads) peak_ffma_kernel(float* out, float a, float b)
{
    float x[kPeakIlp];
#pragma unroll
    for (int i = 0; i < kPeakIlp; ++i) x[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
        for (int i = 0; i < kPeakIlp; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kPeakIlp; ++i) s += x[i];
    if (s == 12345.678f) out[0] = s;
}

// which = 1: FFMA2 (2 ops / lane / instr), broadcast-scalar A operand as in the factored kernel
__global__ void __launch_bounds__(kPeakThreads) peak_ffma2_kernel(float* out, float a, float b)
{
    float2 x[kPeakIlp];
#pragma unroll
    for (int i = 0; i < kPeakIlp; ++i) x[i] = make_float2((float)(threadIdx.x + i), (float)i);
    const float2 bb = make_float2(b, -b);
    for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
        for (int i = 0; i < kPeakIlp; ++i) x[i] = __ffma2_rn(make_float2(a, a), x[i], bb);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kPeakIlp; ++i) s += x[i].x + x[i].y;
    if (s == 12345.678f) out[0] = s;
}

// which = 2: DFMA
__global__ void __launch_bounds__(kPeakThreads) peak_dfma_kernel(double* out, double a, double b)
{
    double x[kPeakIlp];
#pragma unroll
    for (int i = 0; i < kPeakIlp; ++i) x[i] = (double)(threadIdx.x + i);
    for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
        for (int i = 0; i < kPeakIlp; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kPeakIlp; ++i) s += x[i];
    if (s == 12345.678) out[0] = s;
}

// which = 3: MUFU.SIN + MUFU.COS (2 ops / lane / iteration element)
__global__ void __launch_bounds__(kPeakThreads) peak_mufu_kernel(float* out, float a)
{
    float x[kPeakIlp];
#pragma unroll
    for (int i = 0; i < kPeakIlp; ++i) x[i] = a * (float)(threadIdx.x + i);
    for (int it = 0; it < kPeakIters / 4; ++it) {
#pragma unroll
        for (int i = 0; i < kPeakIlp; ++i) {
            float s, c;
            asm volatile("sin.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(x[i]));
            asm volatile("cos.approx.ftz.f32 %0, %1;" : "=f"(c) : "f"(s));
            x[i] = c;
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kPeakIlp; ++i) s += x[i];
    if (s == 12345.678f) out[0] = s;
}

// which = 4: the factored FP32 kernel's inner-loop mix: 32 FFMA2 + 4 LDS.128 per iteration, operands from shared
// memory with the same lane -> address map (lane bit 0 -> group chunk, lane bit 1 -> m chunk).
__global__ void __launch_bounds__(kPeakThreads, 2) peak_mix_kernel(float* out, float a)
{
    __shared__ float4 sA[16 * 32];     // [jj][2 halves][16 gi]
    __shared__ float4 sB[16 * 16];     // [jj][2 halves][8 mi]
    for (int i = threadIdx.x; i < 16 * 32; i += kPeakThreads) sA[i] = make_float4(a, -a, a * 0.5f, 1.f);
    for (int i = threadIdx.x; i < 16 * 16; i += kPeakThreads) sB[i] = make_float4(1.f, a, -a, 0.5f);
    __syncthreads();
    const int lane = threadIdx.x & 31, wq = (threadIdx.x >> 5) & 3;
    const int mi = ((lane >> 1) & 1) | (((lane >> 3) & 3) << 1);
    const int gi = (lane & 1) | (((lane >> 2) & 1) << 1) | (wq << 2);
    float2 acc[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) acc[i] = make_float2(0.f, 0.f);
    for (int it = 0; it < kPeakIters / 16; ++it) {
#pragma unroll 4
        for (int jj = 0; jj < 16; ++jj) {
            const float4 a0 = sA[jj * 32 + gi], a1 = sA[jj * 32 + 16 + gi];
            const float4 p0 = sB[jj * 16 + mi], p1 = sB[jj * 16 + 8 + mi];
            const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            const float2 bv[4] = {make_float2(p0.x, p0.y), make_float2(p0.z, p0.w), make_float2(p1.x, p1.y), make_float2(p1.z, p1.w)};
#pragma unroll
            for (int g = 0; g < 8; ++g)
#pragma unroll
                for (int i = 0; i < 4; ++i) acc[g * 4 + i] = __ffma2_rn(make_float2(av[g], av[g]), bv[i], acc[g * 4 + i]);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 32; ++i) s += acc[i].x + acc[i].y;
    if (s == 12345.678f) out[0] = s;
}

}  // namespace

/*
 * Runs a register-only loop of one instruction class on every SM and returns the measured thread-level operations per second.
 *   which: 0 = FFMA, 1 = FFMA2 (fma.rn.f32x2, counted as 2 FMA per lane), 2 = DFMA, 3 = MUFU.SIN+MUFU.COS (counted
 *          as 2 ops), 4 = FFMA2 with one LDS.128 per 8 (the factored kernel's inner-loop mix)
 * Returns 0 on success (a cudaError_t otherwise) and writes *ops_per_s and *elapsed_ms (HOST, the latter may be NULL).
 */
extern "C" int bench_pipe_peak(int32_t device, int32_t which, double* ops_per_s, double* elapsed_ms)
{
    if (!ops_per_s || which < 0 || which > 4) return (int)cudaErrorInvalidValue;
#define BP_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return (int)e_; } while (0)
    BP_CUDA(cudaSetDevice(device));
    cudaDeviceProp prop;
    BP_CUDA(cudaGetDeviceProperties(&prop, device));
    void* out = nullptr;
    BP_CUDA(cudaMalloc(&out, 64));
    cudaEvent_t e0, e1;
    BP_CUDA(cudaEventCreate(&e0));
    BP_CUDA(cudaEventCreate(&e1));
    const int ctas_per_sm = (which == 4) ? 2 : 4;
    const unsigned grid = (unsigned)(prop.multiProcessorCount * ctas_per_sm * 4);    // 4 full waves
    double ops_per_thread = 0.0;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {                      // rep 0 is the warm-up
        BP_CUDA(cudaEventRecord(e0, 0));
        switch (which) {
            case 0: peak_ffma_kernel<<<grid, kPeakThreads>>>((float*)out, 1.0000001f, 1e-9f);
                    ops_per_thread = (double)kPeakIters * kPeakIlp; break;
            case 1: peak_ffma2_kernel<<<grid, kPeakThreads>>>((float*)out, 1.0000001f, 1e-9f);
                    ops_per_thread = 2.0 * kPeakIters * kPeakIlp; break;
            case 2: peak_dfma_kernel<<<grid, kPeakThreads>>>((double*)out, 1.0000001, 1e-9);
                    ops_per_thread = (double)kPeakIters * kPeakIlp; break;
            case 3: peak_mufu_kernel<<<grid, kPeakThreads>>>((float*)out, 0.001f);
                    ops_per_thread = 2.0 * (kPeakIters / 4) * kPeakIlp; break;
            default: peak_mix_kernel<<<grid, kPeakThreads>>>((float*)out, 0.5f);
                    ops_per_thread = 2.0 * 32.0 * 16.0 * (kPeakIters / 16); break;
        }
        BP_CUDA(cudaGetLastError());
        BP_CUDA(cudaEventRecord(e1, 0));
        BP_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        BP_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0) best_ms = std::min(best_ms, ms);
    }
#undef BP_CUDA
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    *ops_per_s = ops_per_thread * (double)grid * kPeakThreads / (best_ms * 1e-3);
    if (elapsed_ms) *elapsed_ms = best_ms;
    return 0;
}
