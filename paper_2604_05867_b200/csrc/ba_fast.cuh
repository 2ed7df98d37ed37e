// ba_fast.cuh -- BA_MODE_FAST: the deletion transform, position by position.
// Not in the paper; it follows from applying the concatenation identity P:181 one input position at a
// time.  With
//     A_s[y', r] = sum_{x' in {0,1}^s} emb(y', x') p(x'.r),     |y'| <= s, r in {0,1}^{n-s},
// A_0[empty, x] = p(x) and A_n[y, empty] = A(y) = sum_x emb(y,x) p(x).  Reading the next input bit b,
// it is either deleted or kept as the last symbol of y':
//     A_{s+1}[y', r'] = A_s[y', 0.r'] + A_s[y', 1.r']  +  A_s[y'[0:-1], last(y').r']        (forward)
// The input sweep applies the transposed stages to c:  B_n = c,  B_0[empty, x] = sum_y emb(y,x) c(y),
//     B_s[y', b.r'] = B_{s+1}[y', r'] + B_{s+1}[y'.b, r']                                   (backward)
// Stage s is stored as index (code(y') - 1) * 2^{n-s} + r; every stage is < 2^{n+1} doubles.
// These kernels do not enumerate (x,y) terms: throughput quoted for them is "effective terms/s".
#pragma once
#include "ba_internal.h"

// forward stage s -> s+1
__global__ void k_fast_fwd(int n, int s, const double *__restrict__ in, double *__restrict__ out) {
    const int lr = n - s - 1;                                    // bits of r'
    const size_t nout = (((size_t)4 << s) - 1) << lr;            // (2^{s+2}-1) * 2^{lr}
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < nout; o += (size_t)gridDim.x * blockDim.x) {
        const size_t r = o & (((size_t)1 << lr) - 1);
        const uint32_t cy = (uint32_t)(o >> lr) + 1u;           // code(y'), |y'| <= s+1
        const int ly = ba_len_of_code(cy);
        double acc = 0.0;
        if (ly <= s) {
            const size_t base = ((size_t)(cy - 1u) << (lr + 1)) + r;
            acc = in[base] + in[base + ((size_t)1 << lr)];
        }
        if (ly >= 1) {
            const uint32_t cpar = cy >> 1, last = cy & 1u;
            acc += in[((size_t)(cpar - 1u) << (lr + 1)) + ((size_t)last << lr) + r];
        }
        out[o] = acc;
    }
}

// backward stage s+1 -> s
__global__ void k_fast_bwd(int n, int s, const double *__restrict__ in, double *__restrict__ out) {
    const int lr = n - s - 1;                                    // bits of r' (stage s+1)
    const size_t nout = (((size_t)2 << s) - 1) << (lr + 1);      // (2^{s+1}-1) * 2^{lr+1}
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < nout; o += (size_t)gridDim.x * blockDim.x) {
        const size_t rr = o & (((size_t)2 << lr) - 1);           // b.r'
        const uint32_t cy = (uint32_t)(o >> (lr + 1)) + 1u;     // code(y'), |y'| <= s
        const uint32_t b = (uint32_t)(rr >> lr) & 1u;
        const size_t r = rr & (((size_t)1 << lr) - 1);
        const uint32_t cyb = (cy << 1) | b;
        out[o] = in[((size_t)(cy - 1u) << lr) + r] + in[((size_t)(cyb - 1u) << lr) + r];
    }
}
