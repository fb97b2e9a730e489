// mcdc_microbench.cuh -- arithmetic micro-benchmarks behind mcdc_microbench() (include/mcdc.h): measured issue and
// float64 rates of this GPU, the denominators of the ALU roofline bench.py reports beside the HBM one (SURVEY.md
// 8d: "measure FP64 FMA and log/sincos/sqrt/div throughput with a micro-benchmark first").  Every kernel runs
// `iters` trips of a loop with UNROLL independent dependency chains per thread on registers only (no memory), on a
// grid that fills every SM, and folds the chains into one store so that nothing is optimised away.
#pragma once
#include "mcdc_device.cuh"

namespace mcdc {

constexpr int MB_CHAINS = 8;

__global__ void k_mb_ffma(unsigned long long iters, float *out)
{
    float a[MB_CHAINS];
#pragma unroll
    for (int k = 0; k < MB_CHAINS; k++) a[k] = 1.0f + threadIdx.x * 1e-7f + k;
    const float m = 0.9999999f, b = 1e-7f;
    for (unsigned long long i = 0; i < iters; i++) {
#pragma unroll
        for (int k = 0; k < MB_CHAINS; k++) a[k] = fmaf(a[k], m, b);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < MB_CHAINS; k++) s += a[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void k_mb_dfma(unsigned long long iters, double *out)
{
    double a[MB_CHAINS];
#pragma unroll
    for (int k = 0; k < MB_CHAINS; k++) a[k] = 1.0 + threadIdx.x * 1e-9 + k;
    const double m = 0.999999999, b = 1e-9;
    for (unsigned long long i = 0; i < iters; i++) {
#pragma unroll
        for (int k = 0; k < MB_CHAINS; k++) a[k] = fma(a[k], m, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < MB_CHAINS; k++) s += a[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// one library call per chain and trip: 0 log, 1 divide, 2 sqrt, 3 sincospi, 4 reciprocal
template <int OP>
__global__ void k_mb_func(unsigned long long iters, double *out)
{
    constexpr int NC = 4;
    double a[NC];
#pragma unroll
    for (int k = 0; k < NC; k++) a[k] = 0.3 + 0.1 * k + threadIdx.x * 1e-6;
    for (unsigned long long i = 0; i < iters; i++) {
#pragma unroll
        for (int k = 0; k < NC; k++) {
            if (OP == 0) a[k] = 0.5 - 0.03 * log(a[k]);              // stays in (0.4, 0.6)
            else if (OP == 1) a[k] = 0.7 / (a[k] + 0.9);             // stays in (0.3, 0.8)
            else if (OP == 2) a[k] = sqrt(a[k] + 0.2);               // -> fixed point near 1.17
            else if (OP == 3) { double s, c; sincospi(a[k], &s, &c); a[k] = 0.25 + 0.2 * s * c; }
            else a[k] = 1.0 / (a[k] + 1.1);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < NC; k++) s += a[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// one Philox4x32-10 block (= two draws) per chain and trip
__global__ void k_mb_philox(unsigned long long iters, double *out)
{
    constexpr int NC = 4;
    uint32_t c0[NC], c1[NC];
#pragma unroll
    for (int k = 0; k < NC; k++) { c0[k] = threadIdx.x + k; c1[k] = blockIdx.x; }
    for (unsigned long long i = 0; i < iters; i++) {
#pragma unroll
        for (int k = 0; k < NC; k++) {
            uint32_t o0, o1, o2, o3;
            philox4x32_10(c0[k], c1[k], 7u, (uint32_t)i, 1u, 0u, o0, o1, o2, o3);
            c0[k] = o0 ^ o2; c1[k] = o1 ^ o3;
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < NC; k++) s += (double)(c0[k] ^ c1[k]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace mcdc
