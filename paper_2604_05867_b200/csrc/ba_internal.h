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
// LISTS.  The non-empty z are split by their first symbol b (list b); a node carries list b iff b is in its mask.
// A work item of either sweep is a (high part, list) pair: it visits the nodes that carry the list.
//
// CLASSES.  The B_s of a pair depend on the node only through sigma.  Nodes are grouped by their CLASS
// cls = code(y') & (2^BA_KB - 1) (the last BA_KB symbols) and processed in batches of one class, so the
// B_0..B_3 of every pair are constants of the batch.
//
// GROUPS.  Every thread owns, per list, BA_KG groups of BA_GP pair slots.  The pairs of a group share their gathered
// operand (input sweep: one z, up to 4 different v; output sweep: one v, up to 4 different z), which is fetched from
// the staged row ONCE per node (LDS.64) and serves the group's terms; every slot has its own FP64 accumulator, kept
// in a register for the whole work item (static ownership: a slot always belongs to the same (v, z)).  Per term:
//   emb = a0*B0 + a1*B1 [+ a2*B2 + a3*B3]   1-2 IDP.2A (16-bit alphas x 8-bit B's, two products per instruction)
//   acc += (double)emb * operand            exact u32 -> f64 (DADD on the magic number 2^52) + DFMA
// A pair whose chain reaches s = BA_KB under the class (3.4 % of the pairs) is DEEP: its slot holds B = 0 under that
// class and it is handled as a RIDER, one rider per thread: B_0..B_4 static, B_5..B_8 from a direct table indexed by
// the sigma bits 4..7.  When an alpha of the batch does not fit 16 bits (possible for n >= 27 only) the batch runs a
// generic IMAD loop instead.
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
#define BA_KG 4              // groups per thread and list
#define BA_GP 4              // pair slots per group
#define BA_G2_NT 49                     // input sweep: (split, suffix bits, z) targets of the deep part under one class and list
#define BA_NSLOT (BA_KG * BA_GP)
#define BA_KB 4              // class bits
#define BA_NCLS 16           // 2^BA_KB classes
#define BA_ROWB 2048u        // bytes between staged operand rows (2^BA_MLOW doubles)
#define BA_RB_IN 32          // nodes per batch, input sweep (operand half-rows of 2^m doubles)
#define BA_SBR 2             // input sweep: phase-A rounds (of BA_NT nodes) per super-batch
#define BA_RB_OUT 32         // nodes per batch, output sweep (operand rows of 2^m doubles)

struct KConst {                       // passed by value to kernels
    int n, m, h;
    int klen;                         // >= 0: only outputs of this length carry weight (exact channel BDC_{n,k}); -1: all
    double w[BA_NMAX_I + 1];          // w_k = (1-d)^k d^{n-k}                  (NS; R7: 0^0 = 1)
    double lebar[BA_NMAX_I + 1];      // log2( C(n,k) / 2^k ): centring constant of the hoisted log
};

struct NodeRec {                      // 44 bytes, shared memory
    uint32_t a[9];                    // alpha_0..alpha_8 (0 beyond min(k,8))
    uint32_t id;                      // input sweep: code(y') ; output sweep: u
    uint32_t info;                    // mask (bits 0..1) | min(k,8) << 8 | k << 16
};

// A node of a staged batch as the hot loops read it: alphas as 16-bit halves (IDP.2A operands), 48 bytes.
struct BalRec {
    uint32_t a01, a23, a45, a67, a8;  // alpha_0 | alpha_1 << 16, ...; garbage when `big`
    uint32_t big;                     // != 0: an alpha of the node needs more than 16 bits
    uint32_t id;                      // NodeRec::id
    uint32_t node;                    // index of the NodeRec
    double a0d;                       // (double)alpha_0, exact: the type-1 loop (ba_group_loop<1, .>)
    double x0;                        // a per-node operand of the sweep (input sweep: c(y'), the operand of the pair (v, empty))
};
#define BA_BALB 48u

__device__ __forceinline__ BalRec ba_make_bal(const NodeRec &rc, uint32_t node) {
    BalRec bl;
    bl.a01 = rc.a[0] | (rc.a[1] << 16); bl.a23 = rc.a[2] | (rc.a[3] << 16);
    bl.a45 = rc.a[4] | (rc.a[5] << 16); bl.a67 = rc.a[6] | (rc.a[7] << 16);
    bl.a8 = rc.a[8];
    bl.big = (rc.a[0] | rc.a[1] | rc.a[2] | rc.a[3] | rc.a[4] | rc.a[5] | rc.a[6] | rc.a[7]) >> 16;
    bl.id = rc.id; bl.node = node;
    bl.a0d = (double)rc.a[0]; bl.x0 = 0.0;
    return bl;
}

// The schedule of one side, device pointers (host side: GroupSide in ba_tables.h)
struct GroupDev {
    const uint4 *GB;                  // [cls][b][k][tid]
    const uint32_t *GA;               // [b][k][tid]
    const uint16_t *GO;               // [b][k][q][tid]
    const uint16_t *GW;               // [b][warp]: half 0 | half 1 << 8, a half = groups in use | type << 2
    const uint16_t *csr_off;          // [b][nown + 1]
    const uint16_t *csr_idx;          // [b][BA_NSLOT * BA_NT]
    const uint4 *R;                   // riders [cls][b][nr]
    const uint16_t *r_cnt;            // [cls][b]
    const uint16_t *r_csr;            // [cls][b][nown + 1]
    const uint32_t *R8;               // [cls][b][8][nr]: B_4..B_7 by the sigma bits 4..6
    int nr, nown;
    int nsc;                          // schedules (GA, GO, GW, CSR indexed [sc][b]): 2 (sc = class bit 0) or BA_NCLS (sc = class)
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
__device__ __forceinline__ uint2 ba_lds_v2(uint32_t addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 ba_lds_v4(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
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
// TMA-style bulk copy (cp.async.bulk, SASS UBLKCP): `bytes` (a multiple of 16, both addresses 16-byte aligned) from
// global to shared memory by ONE thread; completion is counted in bytes on the mbarrier (complete_tx), which the same
// thread armed with arrive.expect_tx.
__device__ __forceinline__ void ba_mbar_arrive_expect_tx(uint32_t addr, uint32_t bytes) {
    asm volatile("{ .reg .b64 st; mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1; }" ::"r"(addr), "r"(bytes) : "memory");
}
__device__ __forceinline__ void ba_bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t mbar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}

// A lost arrival must fail loudly, not hang the device: trap after ~20 s of SM clocks (far beyond any batch, also
// under a profiler's replay or a preempted context, where a poll count would be reached much sooner than a clock).
// try_wait suspends the warp in hardware until the phase completes or a time limit passes; the common case (the
// phase is already complete, or completes within the first suspensions) costs two instructions.
__device__ __forceinline__ uint32_t ba_mbar_try(uint32_t addr, uint32_t parity) {
    uint32_t done;
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    return done;
}
__device__ __noinline__ void ba_mbar_wait_slow(uint32_t addr, uint32_t parity) {
    const long long t0 = clock64();
    for (;;) {
        for (int i = 0; i < 256; i++) {
            if (ba_mbar_try(addr, parity)) return;
        }
        if (clock64() - t0 > 40000000000ll) __trap();
    }
}
__device__ __forceinline__ void ba_mbar_wait(uint32_t addr, uint32_t parity) {
    if (ba_mbar_try(addr, parity)) return;
    if (ba_mbar_try(addr, parity)) return;
    ba_mbar_wait_slow(addr, parity);
}

// exact uint32 -> FP64 on the FP64 pipe (a DADD on the magic number 2^52) instead of the quarter-rate conversion unit
__device__ __forceinline__ double ba_u2d(uint32_t e) {
    return __hiloint2double(0x43300000, (int)e) - 4503599627370496.0;
}
// Pair slots q of a group whose conversion goes to the conversion unit (I2F.F64.U32, 1 instruction on the otherwise
// idle quarter-rate pipe) instead of the FP64 pipe (MOV + DADD): spreads the per-term conversion over two pipes.
#define BA_CVT_XU_MASK 0x5
template <int Q>
__device__ __forceinline__ double ba_cvt(uint32_t e) {
    if ((BA_CVT_XU_MASK >> Q) & 1) return __uint2double_rn(e);
    return ba_u2d(e);
}

// The hot loop of both sweeps.  A thread's BA_KG groups form two HALVES of two groups; the groups of a half are of one
// TYPE (chosen per warp by the table builder, so a warp mixes a heavy and a light half and all warps carry about the
// same number of instructions per node).  A half loops over the `len` nodes of a batch: Bp = B_0 | B_1<<8 | B_2<<16 |
// B_3<<24 of a slot, rb[k] = shared-memory address of group k's operand in the first staged row, bal = shared-memory
// address of the batch's BalRec array, rows BA_ROWB bytes apart.  K0 = first group of the half, NL = its groups (1, 2).
//   TYPE 4  emb = IDP.2A(a01, B) then IDP.2A(a23, B); exact u32 -> f64; DFMA
//   TYPE 2  no slot of the half ever has B_2 or B_3: one IDP.2A
//   TYPE 1  no slot of the half ever has B_1 (under any class): emb = alpha_0 * B_0 is one product of two integer
//           counts (P:181 with a single split point); the term emb * operand is formed as (alpha_0 * operand) * B_0 with
//           alpha_0 and B_0 converted exactly: one DMUL per group and node, one DFMA per term, no integer work.
template <int TYPE, int K0, int NL>
__device__ __forceinline__ void ba_half_loop(double (&acc)[BA_NSLOT], const uint32_t (&Bp)[BA_NSLOT], const uint32_t (&rb)[BA_KG],
                                             uint32_t bal, int len) {
    if (TYPE == 1) {
        double Bd[NL * BA_GP];
#pragma unroll
        for (int s = 0; s < NL * BA_GP; s++) Bd[s] = (double)(Bp[K0 * BA_GP + s] & 0xffu);
#pragma unroll 4
        for (int i = 0; i < len; i++) {
            const double a0 = ba_lds_f64(bal + (uint32_t)i * BA_BALB + 32u);
#pragma unroll
            for (int k = 0; k < NL; k++) {
                const double t = a0 * ba_lds_f64(rb[K0 + k] + (uint32_t)i * BA_ROWB);
#pragma unroll
                for (int q = 0; q < BA_GP; q++) acc[(K0 + k) * BA_GP + q] = fma(t, Bd[k * BA_GP + q], acc[(K0 + k) * BA_GP + q]);
            }
        }
    } else {
#pragma unroll 4
        for (int i = 0; i < len; i++) {
            uint2 a;
            if (TYPE == 2) { asm volatile("ld.shared.u32 %0, [%1];" : "=r"(a.x) : "r"(bal + (uint32_t)i * BA_BALB)); a.y = 0u; }
            else a = ba_lds_v2(bal + (uint32_t)i * BA_BALB);
#pragma unroll
            for (int k = 0; k < NL; k++) {
                const double op = ba_lds_f64(rb[K0 + k] + (uint32_t)i * BA_ROWB);
#pragma unroll
                for (int q = 0; q < BA_GP; q++) {
                    uint32_t e = __dp2a_lo(a.x, Bp[(K0 + k) * BA_GP + q], 0u);
                    if (TYPE == 4) e = __dp2a_hi(a.y, Bp[(K0 + k) * BA_GP + q], e);
                    const double ed = (q == 0) ? ba_cvt<0>(e) : (q == 1) ? ba_cvt<1>(e) : (q == 2) ? ba_cvt<2>(e) : ba_cvt<3>(e);
                    acc[(K0 + k) * BA_GP + q] = fma(ed, op, acc[(K0 + k) * BA_GP + q]);
                }
            }
        }
    }
}

// The same with the 32-bit alphas of the node records: batches holding an alpha >= 2^16 (n >= 27 only).
// gmask: bit k = group k is in use.
__device__ __forceinline__ void ba_group_loop_wide(double (&acc)[BA_NSLOT], const uint32_t (&Bp)[BA_NSLOT], const uint32_t (&rb)[BA_KG],
                                                   const BalRec *bal, const NodeRec *rec, int len, int gmask) {
    for (int i = 0; i < len; i++) {
        const NodeRec &rc = rec[bal[i].node];
        const uint4 a = make_uint4(rc.a[0], rc.a[1], rc.a[2], rc.a[3]);
#pragma unroll
        for (int k = 0; k < BA_KG; k++) {
            if (!((gmask >> k) & 1)) continue;
            const double op = ba_lds_f64(rb[k] + (uint32_t)i * BA_ROWB);
#pragma unroll
            for (int q = 0; q < BA_GP; q++) {
                const uint32_t bp = Bp[k * BA_GP + q];
                const uint32_t e = a.x * (bp & 0xffu) + a.y * ((bp >> 8) & 0xffu) + a.z * ((bp >> 16) & 0xffu) + a.w * (bp >> 24);
                acc[k * BA_GP + q] = fma(ba_u2d(e), op, acc[k * BA_GP + q]);
            }
        }
    }
}

template <int K0>
__device__ __forceinline__ void ba_half_batch(double (&acc)[BA_NSLOT], const uint32_t (&Bp)[BA_NSLOT], const uint32_t (&rb)[BA_KG],
                                              uint32_t al16, int len, int hm) {
    const int nl = hm & 3, type = hm >> 2;             // half meta: groups in use (0..2) | type << 2
    if (nl == 0) return;
    if (type == 1) { if (nl == 2) ba_half_loop<1, K0, 2>(acc, Bp, rb, al16, len); else ba_half_loop<1, K0, 1>(acc, Bp, rb, al16, len); }
    else if (type == 2) { if (nl == 2) ba_half_loop<2, K0, 2>(acc, Bp, rb, al16, len); else ba_half_loop<2, K0, 1>(acc, Bp, rb, al16, len); }
    else { if (nl == 2) ba_half_loop<4, K0, 2>(acc, Bp, rb, al16, len); else ba_half_loop<4, K0, 1>(acc, Bp, rb, al16, len); }
}

// Dispatch on the warp's static halves (wmeta = half 0 | half 1 << 8) and on whether the batch's alphas fit 16 bits.
__device__ __forceinline__ void ba_group_batch(double (&acc)[BA_NSLOT], const uint32_t (&Bp)[BA_NSLOT], const uint32_t (&rb)[BA_KG],
                                               const BalRec *bal, const NodeRec *rec, int len, int wmeta, bool big) {
    const int h0 = wmeta & 0xff, h1 = (wmeta >> 8) & 0xff;
    if (big) { ba_group_loop_wide(acc, Bp, rb, bal, rec, len, ((1 << (h0 & 3)) - 1) | (((1 << (h1 & 3)) - 1) << 2)); return; }
    const uint32_t al16 = ba_smem_addr(bal);
    ba_half_batch<0>(acc, Bp, rb, al16, len, h0);
    ba_half_batch<2>(acc, Bp, rb, al16, len, h1);
}

// Full chain of a pair with all nine B_s (the pair (v, empty) and the riders): alphas as 16-bit halves
// a01, a23, a45, a67 and alpha_8; B packed B_0..B_3, B_4..B_7, B_8.
__device__ __forceinline__ uint32_t ba_chain9(uint32_t a01, uint32_t a23, uint32_t a45, uint32_t a67, uint32_t a8,
                                              uint32_t b0123, uint32_t b4567, uint32_t b8) {
    uint32_t e = __dp2a_lo(a01, b0123, a8 * b8);
    e = __dp2a_hi(a23, b0123, e);
    e = __dp2a_lo(a45, b4567, e);
    return __dp2a_hi(a67, b4567, e);
}
__device__ __forceinline__ uint32_t ba_chain9_wide(const uint32_t *a, uint32_t b0123, uint32_t b4567, uint32_t b8) {
    return a[0] * (b0123 & 0xffu) + a[1] * ((b0123 >> 8) & 0xffu) + a[2] * ((b0123 >> 16) & 0xffu) + a[3] * (b0123 >> 24) +
           a[4] * (b4567 & 0xffu) + a[5] * ((b4567 >> 8) & 0xffu) + a[6] * ((b4567 >> 16) & 0xffu) + a[7] * (b4567 >> 24) + a[8] * b8;
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
