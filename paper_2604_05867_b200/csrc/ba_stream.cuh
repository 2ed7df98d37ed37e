// ba_stream.cuh -- the streaming kernels of one BA iteration: per-output finish of the output sweep,
// the deterministic second-stage reduction and the normalised update (8(a4)).
#pragma once
#include "ba_internal.h"

// q(y) = w_k A(y) and the gathered operand of the input sweep c(y) = w_k log2( A(y) / ebar_k ),
// A(y) = sum_x emb(y,x) p(x).  ENUM mode: A(y) is the fixed-order sum of the partials the
// output-sweep CTAs own (ba_enum_out.cuh).  FAST mode: A is already complete in `Afull`.
// Writing log2( W/q ) = log2( emb/ebar_k ) - log2( A/ebar_k ) moves the only logarithm that depends on
// the iterate from T(n) terms to 2^{n+1} outputs (SURVEY 7.2 "hoisting the logarithm"); ebar_k =
// C(n,k)/2^k is the mean of emb over a length, which centres both halves.
// c is stored by CODE (c[code(y)] = c[idx(y)+1], entry 0 unused) so that the 2^j outputs y'.z, |z| = j,
// of a prefix y' start at the even index code(y') << j: 16-byte aligned pieces for cp.async.
// crow is the same operand laid out for the input sweep's staging: row (code(y'), b) of 2^m doubles holds c(y'.b.t) at
// position code(t) (z = "b" alone at position b), for every y' of length <= h -- the half row of node y' and list b is
// one contiguous, aligned run (one bulk copy); every c(y) is stored once per split y = y'.z, 1 <= |z| <= m.
__device__ __forceinline__ void ba_store_crow(const KConst &kc, double *__restrict__ crow, uint32_t cy, int k, double v) {
    const int jhi = (k < kc.m) ? k : kc.m;
    for (int j = (k - kc.h > 1) ? (k - kc.h) : 1; j <= jhi; j++) {
        const uint32_t cyp = cy >> j, b = (cy >> (j - 1)) & 1u;
        const uint32_t pos = (j == 1) ? b : ((1u << (j - 1)) | (cy & ((1u << (j - 1)) - 1u)));
        crow[((((size_t)cyp << 1) | b) << kc.m) + pos] = v;
    }
}

__global__ void k_out_final(KConst kc, const double *__restrict__ Apart, const double *__restrict__ Afull,
                            double *__restrict__ q, double *__restrict__ c, double *__restrict__ crow, int sym) {
    const size_t NY = ((size_t)2 << kc.n) - 1;
    const uint32_t NZ = (2u << kc.m) - 1u;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < NY; i += (size_t)gridDim.x * blockDim.x) {
        const uint32_t cy = (uint32_t)(i + 1);
        const int k = ba_len_of_code(cy);
        if (kc.w[k] == 0.0) { q[i] = 0.0; c[i + 1] = 0.0; ba_store_crow(kc, crow, cy, k, 0.0); continue; }   // R7: a length without mass (its partials may be unwritten)
        double A;
        if (Afull) {
            A = Afull[i];
        } else {
            A = 0.0;
            // complement symmetry (sym): A(y) = A(~y); the prefixes with leading symbol 1 were not enumerated
            const uint32_t ce = (sym && k >= 1 && ((cy >> (k - 1)) & 1u)) ? ((1u << k) | (~cy & ((1u << k) - 1u))) : cy;
            const int jlo = (k - kc.h > 0) ? (k - kc.h) : 0;
            const int jhi = (k < kc.m) ? k : kc.m;
            for (int j = jlo; j <= jhi; j++) {       // split y = y'.z, |z| = j
                const uint32_t cyp = ce >> j;
                const uint32_t cz = (1u << j) | (ce & ((1u << j) - 1u));
                A += Apart[(size_t)(cyp - 1u) * NZ + (cz - 1u)];
            }
        }
        const double wk = kc.w[k];
        q[i] = wk * A;
        const double cv = (wk != 0.0) ? wk * (log2(A) - kc.lebar[k]) : 0.0;
        c[i + 1] = cv;
        ba_store_crow(kc, crow, cy, k, cv);
    }
}

// Second stage of the reductions: part holds npart triples {sum p D, max D, sum p 2^D}, one per CTA work
// item of the input sweep.  One block, fixed traversal order => run-to-run bit-reproducible.
// scal[0..2] = I, U, Z ; hist[3*slot..] = I, U, log2 Z.
__global__ void __launch_bounds__(1024) k_finalize(const double *__restrict__ part, size_t npart,
                                                   double *__restrict__ scal, double *__restrict__ hist,
                                                   int slot) {
    __shared__ double s0[1024], s1[1024], s2[1024];
    const int tid = threadIdx.x;
    double a0 = 0.0, a1 = -INFINITY, a2 = 0.0;
    for (size_t i = tid; i < npart; i += 1024) {
        a0 += part[3 * i];
        a1 = fmax(a1, part[3 * i + 1]);
        a2 += part[3 * i + 2];
    }
    s0[tid] = a0; s1[tid] = a1; s2[tid] = a2;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if (tid < o) {
            s0[tid] += s0[tid + o];
            s1[tid] = fmax(s1[tid], s1[tid + o]);
            s2[tid] += s2[tid + o];
        }
        __syncthreads();
    }
    if (tid == 0) {
        scal[0] = s0[0]; scal[1] = s1[0]; scal[2] = s2[0];
        hist[3 * slot] = s0[0]; hist[3 * slot + 1] = s1[0]; hist[3 * slot + 2] = log2(s2[0]);
    }
}

// The low tile on its own: M(u, w) = sum_v p(u.v) emb(w, v) for every high part u and every string w of length <= m
// (stored by code(w), then u: M[code(w) * 2^h + u], row 0 unused -- the out sweep gathers a few w for many nearby u).  With the concatenation identity at the tile boundary,
//     sum_v p(u.v) emb(y', u.v) = sum_s alpha_s M(u, sigma_s),    alpha_s = emb(y'[0:k-s], u), sigma_s = last s symbols of y',
// so the output sweep forms the pair (v, empty) of a node from <= m+1 entries of M instead of 2^m terms and a staged row.
// LT[v][code(w)] = emb(w, v) (bytes).  One block serves four u: every table byte is converted once for four FMAs.
#define BA_LT_UB 4
__global__ void __launch_bounds__(512) k_low_tile(int m, size_t NU, const double *__restrict__ p,
                                                  const uint8_t *__restrict__ LT, double *__restrict__ M) {
    __shared__ double prow[BA_LT_UB << BA_MLOW];
    const int nv = 1 << m, W = 2 << m, tid = threadIdx.x;
    for (size_t u0 = (size_t)blockIdx.x * BA_LT_UB; u0 < NU; u0 += (size_t)gridDim.x * BA_LT_UB) {
        __syncthreads();
        for (int i = tid; i < BA_LT_UB * nv; i += blockDim.x) {
            const size_t uu = u0 + (size_t)(i >> m);
            prow[i] = (uu < NU) ? p[(uu << m) + (size_t)(i & (nv - 1))] : 0.0;
        }
        __syncthreads();
        if (tid < W) {
            double acc[BA_LT_UB];
#pragma unroll
            for (int j = 0; j < BA_LT_UB; j++) acc[j] = 0.0;
#pragma unroll 4
            for (int v = 0; v < nv; v++) {
                const double bd = ba_u2d((uint32_t)LT[(size_t)v * W + tid]);
#pragma unroll
                for (int j = 0; j < BA_LT_UB; j++) acc[j] = fma(bd, prow[j * nv + v], acc[j]);
            }
#pragma unroll
            for (int j = 0; j < BA_LT_UB; j++)
                if (u0 + j < NU) M[(size_t)tid * NU + (u0 + j)] = acc[j];      // by w, then u: the four u of a block fill one sector
        }
    }
}

// p(x) <- max( p(x) 2^{D(x)} / Z, 2^-1000 )    (G8)
__global__ void k_update(size_t NX, double *__restrict__ p, const double *__restrict__ D,
                         const double *__restrict__ scal) {
    const double invZ = 1.0 / scal[2];
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < NX; i += (size_t)gridDim.x * blockDim.x) {
        const double v = p[i] * exp2(D[i]) * invZ;
        p[i] = fmax(v, BA_P_FLOOR);
    }
}

__global__ void k_fill(size_t N, double *__restrict__ a, double v) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) a[i] = v;
}

// Epilogue of the input sweep: D = Hc - (S0 + S1) and the first-stage reductions, one triple per block.
// ENUM mode: S0, S1 are the partial sums of the two lists (ba_enum_in.cuh); FAST mode: S0 is complete, S1 = null.
// sym (complement symmetry, Theorem 4): only x < NX/2 was enumerated; D(~x) = D(x) and p(~x) = p(x) bit for bit,
// so the mirrored half enters the sums by doubling.
__global__ void __launch_bounds__(256) k_in_final(size_t NX, const double *__restrict__ Hc, const double *__restrict__ S0,
                                                  const double *__restrict__ S1, const double *__restrict__ p,
                                                  double *__restrict__ D, double *__restrict__ part, int sym) {
    __shared__ double sr[3 * 8];
    double r0 = 0.0, r1 = -INFINITY, r2 = 0.0;
    // fixed assignment: block b handles the contiguous chunk [b*chunk, (b+1)*chunk)
    const size_t NE = sym ? NX / 2 : NX;
    const size_t chunk = (NE + gridDim.x - 1) / gridDim.x;
    const size_t lo = (size_t)blockIdx.x * chunk, hi = (lo + chunk < NE) ? lo + chunk : NE;
    for (size_t i = lo + threadIdx.x; i < hi; i += blockDim.x) {
        const double Dx = Hc[i] - (S1 ? S0[i] + S1[i] : S0[i]);
        D[i] = Dx;
        const double px = p[i];
        double t0 = px * Dx, t2 = px * exp2(Dx);
        if (sym) { D[NX - 1 - i] = Dx; t0 += t0; t2 += t2; }
        r0 += t0; r1 = fmax(r1, Dx); r2 += t2;
    }
    for (int o = 16; o > 0; o >>= 1) {
        r0 += __shfl_xor_sync(0xffffffffu, r0, o);
        r1 = fmax(r1, __shfl_xor_sync(0xffffffffu, r1, o));
        r2 += __shfl_xor_sync(0xffffffffu, r2, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sr[warp * 3] = r0; sr[warp * 3 + 1] = r1; sr[warp * 3 + 2] = r2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t0 = 0.0, t1 = -INFINITY, t2 = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) { t0 += sr[w * 3]; t1 = fmax(t1, sr[w * 3 + 1]); t2 += sr[w * 3 + 2]; }
        part[(size_t)blockIdx.x * 3] = t0; part[(size_t)blockIdx.x * 3 + 1] = t1; part[(size_t)blockIdx.x * 3 + 2] = t2;
    }
}

// Hc = H_0 + H_1 - K (the two lists of the one-off IN_HC pass; K = an optional constant, 0 when the pass centres term by
// term), mirrored under complement symmetry.
__global__ void k_hc_final(size_t NX, const double *__restrict__ H0, const double *__restrict__ H1, double *__restrict__ Hc, int sym, double K) {
    const size_t NE = sym ? NX / 2 : NX;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < NE; i += (size_t)gridDim.x * blockDim.x) {
        const double v = (H0[i] + H1[i]) - K;
        Hc[i] = v;
        if (sym) Hc[NX - 1 - i] = v;
    }
}
