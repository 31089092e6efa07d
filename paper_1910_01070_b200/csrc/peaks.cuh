// peaks.cuh -- micro-benchmarks behind helios_measure_peaks(): the MEASURED FP32-FMA and MUFU
// rates of this GPU, which the "alu" roofline of bench.py divides by (BASELINE.md "This box":
// "FP32-FMA, MUFU ... peaks are not measured yet -- the build must microbenchmark them"), and the
// dispatch cost of the packed FFMA2 instruction that the cycle budget of the staged kernel rests on
// (DESIGN.md section 6).  Every kernel runs ONE block of 1024 threads per SM (8 warps per scheduler), 8 independent
// dependency chains per thread, no memory traffic inside the loop, about 0.5 ms per kernel, timed with CUDA events;
// block 0 reads clock64() and %globaltimer around its loop, which gives the SM clock the loops ran at.
#pragma once
#include <cuda_runtime.h>

#include "common.cuh"

namespace helios {

constexpr int kPeakIters = 16384;
constexpr int kPeakChains = 8;
constexpr int kPeakThreads = 1024;

enum PeakMode {
    kPeakFfma = 0,          // FFMA  x = x * a + b                    (scalar, 32 FMA per warp instruction)
    kPeakFfma2Scalar = 1,   // FFMA2 x = x * {a,a} + {b,b}            (1 register pair + 2 scalars)
    kPeakFfma2TwoPairs = 2, // FFMA2 x = x * y + {b,b}                (2 register pairs + scalar)
    kPeakFfma2ThreePairs = 3, // FFMA2 x = y * z + x                  (3 distinct register pairs)
    kPeakMufuEx2 = 4,       // MUFU.EX2
    kPeakFfma2PlusAlu = 5,  // 8 FFMA2 (1 pair + 2 scalars) + 8 LOP3 per iteration: does the ALU op ride along?
    kPeakFfma2PlusFsel = 6, // 8 FFMA2 + 8 FSETP/FSEL pairs per iteration
    kPeakFfma3Reg = 7,      // FFMA  x = y * z + x                    (scalar, 3 distinct registers)
    kPeakFfma2PlusMufu = 8, // 8 FFMA2 (1 pair + 2 scalars) + 8 MUFU.EX2 per iteration
    kPeakModes = 9
};

struct PeakTimes {            // written by block 0, thread 0
    long long cycles;         // clock64() across the loop
    long long ns;             // %globaltimer across the loop
};

__device__ __forceinline__ long long global_ns() {
    long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

template <int MODE>
__global__ void __launch_bounds__(kPeakThreads, 1) k_peak(float* out, PeakTimes* times, float a, float b, unsigned m) {
    float2 x[kPeakChains], y[kPeakChains], z[kPeakChains];
    unsigned u[kPeakChains];
#pragma unroll
    for (int j = 0; j < kPeakChains; ++j) {
        x[j] = make_float2(threadIdx.x * 1e-3f + j, threadIdx.x * 2e-3f + j);
        y[j] = make_float2(0.999f + j * 1e-5f + threadIdx.x * 1e-9f, 0.998f + j * 1e-5f);
        z[j] = make_float2(1e-3f * j + threadIdx.x * 1e-9f, 2e-3f * j);
        u[j] = threadIdx.x + j;
    }
    const float2 aa = make_float2(a, a), bb = make_float2(b, b);
    __syncthreads();
    const long long c0 = clock64(), t0 = global_ns();
    for (int i = 0; i < kPeakIters; ++i) {
#pragma unroll
        for (int j = 0; j < kPeakChains; ++j) {
            if (MODE == kPeakFfma) { x[j].x = fmaf(x[j].x, a, b); }
            if (MODE == kPeakFfma2Scalar || MODE == kPeakFfma2PlusAlu || MODE == kPeakFfma2PlusFsel || MODE == kPeakFfma2PlusMufu)
                x[j] = __ffma2_rn(x[j], aa, bb);
            if (MODE == kPeakFfma3Reg) x[j].x = fmaf(y[j].x, z[j].x, x[j].x);
            if (MODE == kPeakFfma2TwoPairs) x[j] = __ffma2_rn(x[j], y[j], bb);
            if (MODE == kPeakFfma2ThreePairs) x[j] = __ffma2_rn(y[j], z[j], x[j]);
            if (MODE == kPeakMufuEx2) { float r; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x[j].x)); x[j].x = r; }
        }
        if (MODE == kPeakFfma2PlusAlu) {
#pragma unroll
            for (int j = 0; j < kPeakChains; ++j) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[j]) : "r"(m), "r"(i));
        }
        if (MODE == kPeakFfma2PlusMufu) {
#pragma unroll
            for (int j = 0; j < kPeakChains; ++j) { float r; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(z[j].x)); z[j].x = r; }
        }
        if (MODE == kPeakFfma2PlusFsel) {
#pragma unroll
            for (int j = 0; j < kPeakChains; ++j)
                asm volatile("{ .reg .pred p; setp.lt.f32 p, %0, %1; selp.f32 %0, %2, %0, p; }" : "+f"(z[j].x) : "f"(y[j].x), "f"(y[j].y));
        }
    }
    __syncthreads();
    const long long c1 = clock64(), t1 = global_ns();
    float s = 0.0f;
#pragma unroll
    for (int j = 0; j < kPeakChains; ++j) s += x[j].x + x[j].y + y[j].x + z[j].x + (float)u[j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (blockIdx.x == 0 && threadIdx.x == 0) { times->cycles = c1 - c0; times->ns = t1 - t0; }
}

}  // namespace helios
