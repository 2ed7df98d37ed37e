// ba_peaks.cuh -- in-library microbenchmarks of the pipes the ENUM sweeps use ("the bench must measure
// both peaks with its own microbenchmarks in the same run").  Each kernel runs a dependence-free stream of ONE
// instruction kind on every SM (one 512-thread CTA per SM, 16 warps, 8 independent chains per thread) and reports
// warp-instructions per clock per SM from clock64(); the SM clock comes from the same kernels timed with CUDA events.
//   PK_DFMA   FP64 fused multiply-add, two register operand pairs        (the per-term DFMA / DADD pipe)
//   PK_IDP    IDP.2A (16-bit x 8-bit dot product, the emb combine)        (the integer multiply pipe, shared with IMAD)
//   PK_LDS64  conflict-free LDS.64, one operand per lane                  (the gathered operand)
//   PK_FFMA   FP32 fused multiply-add (both FMA pipes): the issue rate of a scheduler, one warp-instruction per clock
#pragma once
#include "ba_internal.h"

enum { PK_DFMA = 0, PK_IDP = 1, PK_LDS64 = 2, PK_FFMA = 3, PK_N = 4 };

template <int KIND>
__global__ void __launch_bounds__(512, 1) k_peak(unsigned long long *clk, double *sink, int iters, unsigned seed) {
    __shared__ double sm[2048];
    const int tid = threadIdx.x;
    for (int i = tid; i < 2048; i += blockDim.x) sm[i] = 1.0 + i * 1e-9;
    __syncthreads();
    unsigned a[8];
    double d[8];
    float f[8];
#pragma unroll
    for (int j = 0; j < 8; j++) { a[j] = seed * (j + 1) + tid; d[j] = 1.0 + j + tid * 1e-6; f[j] = 1.0f + j; }
    const unsigned b = seed | 0x01010101u, c2 = seed * 7 + 3;
    const double m1 = 1.0 + seed * 1e-12, m2 = seed * 1e-15;
    const uint32_t sbase = ba_smem_addr(sm) + (uint32_t)(tid & 31) * 8u;
    const long long t0 = clock64();
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 4; r++)
#pragma unroll
            for (int j = 0; j < 8; j++) {
                if (KIND == PK_DFMA) d[j] = fma(d[j], m1, m2);
                if (KIND == PK_IDP) a[j] = __dp2a_lo(a[j], b, c2);
                if (KIND == PK_LDS64) d[j] += ba_lds_f64(sbase + (uint32_t)((j + r * 8) * 256));
                if (KIND == PK_FFMA) f[j] = fmaf(f[j], 1.0001f, 0.5f);
            }
    }
    const long long t1 = clock64();
    double s = 0;
    unsigned u = 0;
    float ff = 0;
#pragma unroll
    for (int j = 0; j < 8; j++) { s += d[j]; u += a[j]; ff += f[j]; }
    if (s == 123.456 || u == 77u || ff == 3.25f) sink[0] = s + u + ff;      // keeps the chains alive
    if (tid == 0) clk[blockIdx.x] = (unsigned long long)(t1 - t0);
}
