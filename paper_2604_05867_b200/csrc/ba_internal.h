// ba_internal.h -- shared declarations of libba's kernels (not part of the C ABI).
//
// Decomposition used by every ENUM kernel: x = u.v with |u| = h = n-m high bits
// and |v| = m = min(n, BA_MLOW) low bits, x = (u << m) | v.  A string s of length L and MSB-first
// value val is carried as code(s) = (1 << L) | val, so idx(s) = code(s) - 1 (include/ba.h layout) and
// code(s.t) = (code(s) << |t|) | val(t).  The concatenation identity of P:181,
//   emb(y, u.v) = sum_t emb(y[0:t], u) * emb(y[t:], v),
// lets the low m positions be served by a small table of the m-bit deletion channel ("low table").
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#define BA_MLOW 8            // low-tile width m (bits); 2^m threads per CTA in the ENUM kernels
#define BA_NMAX_I 30
#define BA_HIST_CAP 65536    // ring of per-iteration {I, U, log2 Z}
#define BA_LINK_NONE 127u
#define BA_P_FLOOR 9.3326361850321888e-302   // 2^-1000 (G8)

// Low-table entry word for (v, z), z a distinct subsequence of the m-bit string v:
//   bits  0..8   code(z)              (<= 2^{m+1}-1 = 511)
//   bits  9..15  B = emb(z, v)        (<= C(8,4) = 70)
//   bits 16..22  local index of (0.z) in v's list, or BA_LINK_NONE
//   bits 23..29  local index of (1.z) in v's list, or BA_LINK_NONE
// v's list is ordered [empty][z starting with 0][z starting with 1].
// vinfo[v] = base (bits 0..13) | n0 << 14 (7 bits) | n1 << 21 (7 bits).
__host__ __device__ __forceinline__ uint32_t lt_code(uint32_t w) { return w & 511u; }
__host__ __device__ __forceinline__ uint32_t lt_B(uint32_t w) { return (w >> 9) & 127u; }
__host__ __device__ __forceinline__ uint32_t lt_link(uint32_t w, uint32_t b) { return (w >> (16 + 7 * b)) & 127u; }
__host__ __device__ __forceinline__ uint32_t vi_base(uint32_t vi) { return vi & 0x3fffu; }
__host__ __device__ __forceinline__ uint32_t vi_n0(uint32_t vi) { return (vi >> 14) & 127u; }
__host__ __device__ __forceinline__ uint32_t vi_n1(uint32_t vi) { return (vi >> 21) & 127u; }

// Per-thread entry of the output-sweep assignment list (16 bit): v (bits 0..7) | local index of z in
// v's list (bits 8..14) | valid (bit 15).
__host__ __device__ __forceinline__ uint32_t tl_v(uint32_t e) { return e & 255u; }
__host__ __device__ __forceinline__ uint32_t tl_el(uint32_t e) { return (e >> 8) & 127u; }
__host__ __device__ __forceinline__ bool tl_valid(uint32_t e) { return (e >> 15) & 1u; }

struct KConst {                       // passed by value to kernels
    int n, m, h;
    double w[BA_NMAX_I + 1];          // w_k = (1-d)^k d^{n-k}                  (NS; R7: 0^0 = 1)
    double lebar[BA_NMAX_I + 1];      // log2( C(n,k) / 2^k ): centring constant of the hoisted log
};

// number of slots of class j (outputs z of length j) per thread in the output-sweep assignment
struct OutLayout {
    int slots[BA_MLOW + 1];
    int off[BA_MLOW + 2];             // prefix sums; off[m+1] = total slots
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
