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
//   emb(y'.z, u.v) = sum_{s>=0} alpha_s * B_s,   B_s = B(sigma_s.z, v) = emb(sigma_s.z, v),
// sigma_s = last s symbols of y'.  B_s = 0 implies B_{s+1} = 0, and B_s = 0 for s > m - |z|.
//
// CLASSES.  The B_s of a pair depend on the node only through sigma.  Nodes are grouped by their CLASS
// cls = code(y') & (2^BA_KB - 1) (the last BA_KB symbols) and processed in runs of one class, so the
// B_0..B_3 of every pair are constants of the run: each thread loads the BA_C pairs of a chunk once
// (class-specific FAST table, global memory / L2) and then loops over the nodes of the run with
//   emb = a0*B0 + a1*B1 + a2*B2 + a3*B3        (4 IMAD, no unpacking, no links, no votes)
// A pair whose chain reaches s = BA_KB under the class (3.4 % of the pairs) is DEEP: it is left out of
// the class's fast table and handled as a RIDER, one rider per thread: B_0..B_4 static, B_5..B_8 from a
// direct table indexed by the sigma bits 4..7.
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
#define BA_C 5               // pairs per chunk
#define BA_NC 3              // chunk slots per thread and list
#define BA_KB 4              // class bits
#define BA_NCLS 16           // 2^BA_KB classes
#define BA_RB_IN 32          // nodes per batch, input sweep (operand half-rows of 2^m doubles)
#define BA_SBR 3             // input sweep: phase-A rounds (of BA_NT nodes) per super-batch
#define BA_RB_OUT 32         // nodes per batch, output sweep (operand rows of 2^m doubles)

// ---- v-major prepend links Wv (host side only: the table builder walks them; the kernels read the direct
// tables EPS8 / RI8 / RO8 instead): one uint32 per entry of v's list ([0] null, [1] empty string, then the
// non-empty subsequences of v):  W = l0 | cB0 << 8 | l1 << 16 | cB1 << 24,  l_b = local index of b.z in
// v's list (0 = null: b.z is not a subsequence of v), cB_b = B(b.z, v).
// ---- fast pairs: uint2 {B0 | B1<<8 | B2<<16 | B3<<24, byte offset of the operand in the staged row}
//   [class][list b][slot c][pair q][thread]; slot (b,c,thread) always belongs to the same v (input sweep)
//   or z (output sweep), so its FP64 accumulator lives in a register for the whole work item.  Within a
//   half-warp the offsets of one (class,b,c,q) are dealt to distinct 8-byte bank pairs where possible.
// ---- riders: uint4 {B0..B3, B4 | link4 << 8 | owner << 16, row byte offset, byte offset of v's list in Wv}

struct KConst {                       // passed by value to kernels
    int n, m, h;
    int klen;                         // >= 0: only outputs of this length carry weight (exact channel BDC_{n,k}); -1: all
    double w[BA_NMAX_I + 1];          // w_k = (1-d)^k d^{n-k}                  (NS; R7: 0^0 = 1)
    double lebar[BA_NMAX_I + 1];      // log2( C(n,k) / 2^k ): centring constant of the hoisted log
};

struct NodeRec {                      // 48 bytes, shared memory
    uint32_t a[9];                    // alpha_0..alpha_8 (0 beyond min(k,8))
    uint32_t id;                      // input sweep: code(y') ; output sweep: u
    uint32_t info;                    // mask (bits 0..1) | min(k,8) << 8 | k << 16
    uint32_t pad;
};

// Position of operand number `pos` in a staged row: bits 1..3 are XORed with bits 4..6, so that operands
// whose numbers agree in the low four bits (the strings sharing their last symbols) spread over the 8-byte bank
// pairs.  An involution that keeps the two operands of a 16-byte piece together.
__host__ __device__ __forceinline__ uint32_t ba_swz(uint32_t pos) { return pos ^ (((pos >> 4) & 7u) << 1); }

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

// ---- mbarrier ring (shared-memory transaction barriers): the batches' operand rows are produced by all
// threads with cp.async and consumed by all threads; a FULL barrier per stage completes when every thread's
// copies for that stage have landed (cp.async.mbarrier.arrive), an EMPTY barrier when every thread has finished
// reading it.  Warps meet only through these barriers, so they may drift by a batch instead of stopping at a
// CTA-wide barrier after every batch.
__device__ __forceinline__ void ba_mbar_init(uint32_t addr, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(addr), "r"(count) : "memory");
}
__device__ __forceinline__ void ba_mbar_arrive(uint32_t addr) {
    asm volatile("{ .reg .b64 st; mbarrier.arrive.shared::cta.b64 st, [%0]; }" ::"r"(addr) : "memory");
}
__device__ __forceinline__ void ba_mbar_arrive_on_copies(uint32_t addr) {      // arrives when this thread's cp.async landed
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(addr) : "memory");
}
__device__ __forceinline__ void ba_mbar_wait(uint32_t addr, uint32_t parity) {
    uint32_t done = 0;
    for (uint32_t spin = 0; !done; spin++) {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(addr), "r"(parity) : "memory");
        if (spin > (1u << 26)) __trap();                    // a lost arrival must fail loudly, not hang the device
    }
}

// exact uint32 -> FP64 on the FP64 pipe (a DADD) instead of the quarter-rate conversion unit
__device__ __forceinline__ double ba_u2d(uint32_t e) {
    return __hiloint2double(0x43300000, (int)e) - 4503599627370496.0;
}

// Pair positions q of a chunk whose int->FP64 conversion goes to the conversion unit (I2F on the XU pipe)
// instead of the FP64 pipe: spreads the per-term conversion over two otherwise idle/half-rate pipes.
#ifndef BA_CVT_XU_MASK
#define BA_CVT_XU_MASK 0x0a
#endif
template <int Q>
__device__ __forceinline__ double ba_cvt(uint32_t e) {
    if ((BA_CVT_XU_MASK >> Q) & 1) return __uint2double_rn(e);
    return ba_u2d(e);
}

// The hot loop of both sweeps: the BA_C pairs of one chunk (bp = B_0 | B_1<<8 | B_2<<16 | B_3<<24, ad = byte
// offset of the operand in a staged row) against the `len` nodes of a batch (bal[i] = alpha_0..3, operand
// rows at rowbase + i*ROWB).  NS = number of B_s that can be non-zero in this warp's pairs (depth + 1).
template <int NS>
__device__ __forceinline__ double ba_fast_loop(double s, const uint4 *bal, uint32_t rowbase, uint32_t ROWB, int len,
                                               const uint32_t (&bp)[BA_C], const uint32_t (&ad)[BA_C]) {
    uint32_t B0[BA_C], B1[BA_C], B2[BA_C], B3[BA_C];
#pragma unroll
    for (int q = 0; q < BA_C; q++) {
        B0[q] = bp[q] & 0xffu; B1[q] = (bp[q] >> 8) & 0xffu; B2[q] = (bp[q] >> 16) & 0xffu; B3[q] = bp[q] >> 24;
    }
    double s2 = 0.0;                                        // two dependent-FMA chains instead of one
#pragma unroll 2
    for (int i = 0; i < len; i++) {
        const uint4 al = bal[i];
        const uint32_t rb = rowbase + (uint32_t)i * ROWB;
#pragma unroll
        for (int q = 0; q < BA_C; q++) {
            uint32_t emb = al.x * B0[q];
            if (NS >= 2) emb += al.y * B1[q];
            if (NS >= 3) emb += al.z * B2[q];
            if (NS >= 4) emb += al.w * B3[q];
            const double e = (q == 0) ? ba_cvt<0>(emb) : (q == 1) ? ba_cvt<1>(emb) : (q == 2) ? ba_cvt<2>(emb)
                           : (q == 3) ? ba_cvt<3>(emb) : ba_cvt<4>(emb);
            if (q & 1) s2 = fma(e, ba_lds_f64(rb + ad[q]), s2);
            else s = fma(e, ba_lds_f64(rb + ad[q]), s);
        }
    }
    return s + s2;
}

// Dispatch on the warp-uniform depth of the chunk (B_s = 0 implies B_{s+1} = 0).
__device__ __forceinline__ double ba_fast_chunk(double s, const uint4 *bal, uint32_t rowbase, uint32_t ROWB, int len,
                                                const uint32_t (&bp)[BA_C], const uint32_t (&ad)[BA_C]) {
    uint32_t any = 0;
#pragma unroll
    for (int q = 0; q < BA_C; q++) any |= bp[q];
    any = __reduce_or_sync(0xffffffffu, any);
    if (!any) return s;                                     // no pair of this warp in the slot
    if (any >> 24) return ba_fast_loop<4>(s, bal, rowbase, ROWB, len, bp, ad);
    if (any >> 16) return ba_fast_loop<3>(s, bal, rowbase, ROWB, len, bp, ad);
    if (any >> 8) return ba_fast_loop<2>(s, bal, rowbase, ROWB, len, bp, ad);
    return ba_fast_loop<1>(s, bal, rowbase, ROWB, len, bp, ad);
}

// Stable rank of every thread's key among the CTA (keys < NKEY; key < 0 = not ranked): order[pos] = tid with
// pos = start[key] + (number of lower tids with the same key).  wcnt: [BA_NT/32][NKEY] scratch, start: [NKEY+1].
template <int NKEY>
__device__ __forceinline__ void ba_bucket_sort(int key, uint16_t *order, uint16_t *wcnt, uint16_t *start) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < (BA_NT / 32) * NKEY; i += BA_NT) wcnt[i] = 0;
    __syncthreads();
    const unsigned mm = __match_any_sync(0xffffffffu, key);
    const int rank = __popc(mm & ((1u << lane) - 1u));
    if (key >= 0 && rank == 0) wcnt[warp * NKEY + key] = (uint16_t)__popc(mm);
    __syncthreads();
    if (tid < NKEY) {                                       // exclusive scan over the warps, per key
        int run = 0;
        for (int w = 0; w < BA_NT / 32; w++) { const int c = wcnt[w * NKEY + tid]; wcnt[w * NKEY + tid] = (uint16_t)run; run += c; }
        start[tid + 1] = (uint16_t)run;                     // bucket sizes, scanned below
    }
    __syncthreads();
    if (tid == 0) {
        int run = 0;
        start[0] = 0;
        for (int k = 0; k < NKEY; k++) { const int c = start[k + 1]; start[k + 1] = (uint16_t)(run + c); run += c; }
    }
    __syncthreads();
    if (key >= 0) order[start[key] + wcnt[warp * NKEY + key] + rank] = (uint16_t)tid;
    __syncthreads();                                        // order[] complete; wcnt may be reused
}
