// ba_internal.h -- shared declarations of libba's kernels (not part of the C ABI).
//
// Tiling used by every ENUM kernel: x = u.v with |u| = h = n-m high bits and
// |v| = m = min(n, BA_MLOW) low bits, x = (u << m) | v.  A string s of length L and MSB-first value
// val is carried as code(s) = (1 << L) | val, so idx(s) = code(s) - 1 (include/ba.h layout) and
// code(s.t) = (code(s) << |t|) | val(t).  The concatenation identity of P:181,
//   emb(y, u.v) = sum_t emb(y[0:t], u) * emb(y[t:], v),
// lets the low m positions be served by a static table of the m-bit deletion channel ("low table").
//
// A NODE is a pair (u, y') with y' a subsequence of u (|y'| = k).  Its record carries
//   alpha_s = emb(y'[0:k-s], u), s = 0..min(k,m)      (integer DP of P:173 / P:260-274 on u)
//   sigma   = the last min(k,8) symbols of y'          (low bits of code(y'))
//   mask    = which symbols b cannot follow y' in u after its leftmost embedding (NextPos)
// The (x,y) terms of the node are the PAIRS (v, z), z a subsequence of v with z empty or z[0] in mask:
// y = y'.z is then visited at exactly one node (y' = the longest prefix of y embeddable in u), and
//   emb(y'.z, u.v) = sum_{s>=0} alpha_s * B(sigma_s.z, v),   B(w, v) = emb(w, v),
// sigma_s = last s symbols of y'.  The sum is a CHAIN of "prepend" links in v's list of subsequences.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#define BA_MLOW 8            // low-tile width m (bits)
#define BA_NMAX_I 30
#define BA_HMAX 22           // BA_NMAX_I - BA_MLOW: longest high part
#define BA_HIST_CAP 65536    // ring of per-iteration {I, U, log2 Z}
#define BA_P_FLOOR 9.3326361850321888e-302   // 2^-1000 (G8)

#define BA_NT 512            // threads per CTA of the ENUM kernels (one CTA per SM)
#define BA_C 5               // pairs per chunk (odd: consecutive chunks are bank-conflict free)
#define BA_NC 3              // chunk slots per thread and list
#define BA_GRP 4             // nodes per barrier group
#define BA_NSTAGE 8          // staged rows (2 groups)

// ---- low table, v-major ("T64"): one uint2 {W, P} per entry -------------------------------------
// v's list: [0] null  [1] empty string  [2 ..) z starting with 0, longest first, zero-padded to a
// multiple of BA_C   [..) z starting with 1, likewise.  For the entry of (v, z):
//   W = l0 | cB0 << 8 | l1 << 16 | cB1 << 24   l_b = local index of b.z in v's list (0 = null: b.z is
//                                              not a subsequence of v), cB_b = B(b.z, v)
//   P = B(z,v) | |z| << 8 | (8 * code(z)) << 16     (8*code(z) = byte offset in a staged row)
// The null entry and the padding are all-zero words: emb = 0, links stay on null.
// ---- z-major table ("Tz"), output sweep: for each z its supersequences v, ascending, zero-padded
//   W as above;  P' = B(z,v) | v << 8 | (4 * vbase[v]) << 16   (byte offset of v's list in Wv)
// ---- chunk descriptors: uint2 per (list b, slot, thread)
//   in : x = byte offset of the chunk's first pair in T64 | v << 20 | valid << 31 ; y = byte offset of v's list
//   out: x = byte offset of the chunk's first pair in Tz  | code(z) << 20 | valid << 31 ; y = 0

struct KConst {                       // passed by value to kernels
    int n, m, h;
    double w[BA_NMAX_I + 1];          // w_k = (1-d)^k d^{n-k}                  (NS; R7: 0^0 = 1)
    double lebar[BA_NMAX_I + 1];      // log2( C(n,k) / 2^k ): centring constant of the hoisted log
};

struct NodeRec {                      // 48 bytes, shared memory
    uint32_t a[9];                    // alpha_0..alpha_8 (0 beyond min(k,8))
    uint32_t id;                      // input sweep: code(y') ; output sweep: u
    uint32_t info;                    // mask (bits 0..1) | min(k,8) << 8 | k << 16
    uint32_t pad;
};

__device__ __forceinline__ int ba_len_of_code(uint32_t code) { return 31 - __clz(code); }

// First position p >= from (paper positions, 0 = leftmost) with bit b in the L-bit string s, or L.
__device__ __forceinline__ int ba_nextpos(uint32_t s, int L, int from, uint32_t b) {
    if (from >= L) return L;
    uint32_t t = b ? s : ~s;
    t &= (L - from >= 32) ? 0xffffffffu : ((1u << (L - from)) - 1u);
    if (t == 0) return L;
    return L - 1 - (31 - __clz(t));
}

// ---- shared-memory and async-copy primitives ---------------------------------------------------
__device__ __forceinline__ uint32_t ba_smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t ba_lds_u16(uint32_t addr) {
    uint16_t v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
    return (uint32_t)v;
}
__device__ __forceinline__ uint2 ba_lds_v2(uint32_t addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ double ba_lds_f64(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void ba_cp_async16(uint32_t dst, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void ba_cp_async8(uint32_t dst, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void ba_cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// exact uint32 -> FP64 on the FP64 pipe (a DADD) instead of the quarter-rate conversion unit
__device__ __forceinline__ double ba_u2d(uint32_t e) {
    return __hiloint2double(0x43300000, (int)e) - 4503599627370496.0;
}

// Chain steps S = 2..8 for CN pairs at once: lk[i] = local index of sigma_{S-1}.z in its v's list,
// vb[i] = shared byte address of that list's W words (stride STRIDE bytes).  L = min(k,8) is uniform
// over the CTA; the vote ends the walk as soon as every lane of the warp sits on null entries.
template <int S, int CN, int STRIDE>
struct BaChain {
    static __device__ __forceinline__ void run(uint32_t (&emb)[CN], uint32_t (&lk)[CN], const uint32_t (&vb)[CN],
                                               uint32_t anyl, const uint32_t (&al)[9], uint32_t sig, int L) {
        if (L >= S && __any_sync(0xffffffffu, anyl != 0u)) {
            const uint32_t bo = ((sig >> (S - 1)) & 1u) * 2u;
            anyl = 0u;
#pragma unroll
            for (int i = 0; i < CN; i++) {
                const uint32_t hw = ba_lds_u16(vb[i] + bo + lk[i] * (uint32_t)STRIDE);
                emb[i] += al[S] * (hw >> 8);
                lk[i] = hw & 0xffu;
                anyl |= lk[i];
            }
            BaChain<S + 1, CN, STRIDE>::run(emb, lk, vb, anyl, al, sig, L);
        }
    }
};
template <int CN, int STRIDE>
struct BaChain<9, CN, STRIDE> {
    static __device__ __forceinline__ void run(uint32_t (&)[CN], uint32_t (&)[CN], const uint32_t (&)[CN], uint32_t,
                                               const uint32_t (&)[9], uint32_t, int) {}
};

// The same walk for one pair without warp votes (lanes of a warp may belong to different nodes).
template <int STRIDE>
__device__ __forceinline__ uint32_t ba_chain_single(uint32_t W, uint32_t B, uint32_t vb, const uint32_t (&al)[9],
                                                    uint32_t sig, int L) {
    uint32_t emb = al[0] * B;
    if (L >= 1) {
        uint32_t hw = (sig & 1u) ? (W >> 16) : (W & 0xffffu);
        emb += al[1] * (hw >> 8);
        uint32_t lk = hw & 0xffu;
#pragma unroll
        for (int s = 2; s <= 8; s++) {
            if (L >= s && lk != 0u) {
                hw = ba_lds_u16(vb + ((sig >> (s - 1)) & 1u) * 2u + lk * (uint32_t)STRIDE);
                emb += al[s] * (hw >> 8);
                lk = hw & 0xffu;
            }
        }
    }
    return emb;
}
