// ba_enum_in.cuh -- input sweep: for every x, enumerate its distinct subsequences y
// with their integer embedding counts emb(y,x) exactly once each.
//
// Work item = a high part u (h bits) with its 2^m inputs x = u.v; one persistent CTA per SM takes
// items from an atomic counter.  Per item, in super-batches of BA_SBR * BA_NT nodes:
//   phase A  (BA_SBR rounds) every thread UNRANKS one node per round: the r-th distinct subsequence y' of
//            u in trie pre-order (the paper's stringUnrank idea, Alg. 4, with the subtree sizes
//            Sub[pos] in the role of the Count table P:260-274 and NextPos P:256-258 done with clz on bit
//            masks), and carries the integer embedding-count DP  E[i] = emb(y', u[0:i])  in registers
//            along the descent; the node record {alpha_0..8, code(y'), mask} goes to shared memory.
//   eps      the pair (v, empty) of every node of the round: thread (v, node), all nine B(sigma_s, v) from
//            one 8-byte read of the direct table EPS8[sigma_8][v].
//   sort     per list b (non-empty z starting with b; a node carries list b iff b cannot follow y' in u)
//            the nodes are ranked, stably, by class; the rounds' runs are merged into one order.
//   phase B  batches of <= BA_RB_IN nodes of one (list, class).  The operands c(y'.z), z = b.t, of a node
//            form a HALF ROW of 2^m doubles indexed by code(t) (8 contiguous segments of c), staged with
//            16-byte cp.async, double buffered.  Every thread owns BA_NC chunks of BA_C pairs (v,z) per
//            list; the chunk's B_0..B_3 and row offsets are constants of the batch (ba_internal.h
//            "CLASSES"), so the loop over the nodes of the batch costs, per (x,y) term,
//                 1-4 IMAD (emb) + 1 LDS.64 (operand) + 1 exact u32->f64 + 1 DFMA
//            with one FP64 accumulator per chunk kept in a register for the whole item.  Deep pairs
//            ride along, one per thread, their partial sums handed to thread v through shared memory
//            in a fixed order.
//   epilogue thread v adds the accumulators of v's chunks in a fixed order: D(x) = Hc(x) - sum_y emb c(y).
// MODE:
//   IN_SWEEP  D(x) and the fused reductions of 8(a3) (sum p D, max D, sum p 2^D per item)
//   IN_HC     Hc(x) = sum_y w_k emb log2(emb/ebar_k)   (iteration independent; built once per ctx)
//   IN_DEBUG  emb_out[idx(y)] = emb(y,x) for one x     (ba_debug_emb_row)
//   IN_COUNT  number of visited terms and sum of emb   (ba_debug_count_terms)
#pragma once
#include "ba_internal.h"

enum { IN_SWEEP = 0, IN_HC = 1, IN_DEBUG = 2, IN_COUNT = 3 };

#define BA_IN_SB (BA_SBR * BA_NT)                           // nodes per super-batch
#define BA_IN_NBKT (2 * BA_NCLS)                            // buckets: list b, class
#define BA_IN_MAXB (BA_IN_NBKT + 2 * BA_IN_SB / BA_RB_IN)

struct InArgs {
    KConst kc;
    const uint2 *EPS8;        // [256][2^m]: B(sigma_s, v), s = 1..8, of the pair (v, empty)
    const uint32_t *RI8;      // [cls][b][16][nri]: B_5..B_8 of a rider by the sigma bits 4..7
    const uint2 *FI;          // fast pairs [cls][b][c][q][tid]; .y = 8 * code(z[1:])
    const uint4 *RI;          // riders [cls][b][nri]
    const uint16_t *ri_cnt;   // [cls][b]
    const uint16_t *ri_csr;   // [cls][b][2^m + 1]
    int nri;
    const uint16_t *owner;    // [b][c][tid] -> v
    const uint16_t *csr_off;  // [2^m + 1]
    const uint16_t *csr_idx;
    int ncsr;
    const double *c;          // IN_SWEEP: c[code(y)], 2^{n+1} entries (entry 0 unused)
    const double *p;          // IN_SWEEP: p(x)
    double *Hc;               // IN_HC: out; IN_SWEEP: in
    double *D;                // IN_SWEEP: out
    double *part;             // IN_SWEEP: 3 doubles per u: sum p D, max D, sum p 2^D
    unsigned int *counter;    // work counter (zeroed before launch)
    int sym;                  // 1: p(x) = p(~x) (Theorem 4): only the u with leading bit 0 are enumerated, D is mirrored
    uint32_t dbg_x;           // IN_DEBUG
    uint32_t *dbg_out;        // IN_DEBUG: NY zero-filled
    unsigned long long *cnt;  // IN_COUNT: [0] terms, [1] emb sum
};

struct InSmem { size_t rec, ceps, rows, bal, bnode, ordr, seg, order, gstart, wcnt, batch, rsum, csr_off, sub, red, kcw, item, total; };

__host__ __device__ static inline InSmem enum_in_smem(int m, int ncsr, int nri) {
    InSmem s;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 15) & ~(size_t)15; return at; };
    s.rec = take((size_t)BA_IN_SB * sizeof(NodeRec));
    {                                                      // c(y') of a round (phase A / eps) and the rider sums
        const size_t ce = (size_t)BA_NT * 8, rs = (size_t)2 * 2 * nri * 8;   // of phase B share one area
        s.ceps = take(ce > rs ? ce : rs);
        s.rsum = s.ceps;
    }
    size_t rows = (size_t)2 * BA_RB_IN * ((size_t)1 << m) * 8, ac = ((size_t)2 * BA_NC + 2) * BA_NT * 8;
    s.rows = take(rows > ac ? rows : ac);                  // the epilogue's accumulator staging aliases the rows
    s.bal = take((size_t)2 * BA_RB_IN * 16);
    s.bnode = take((size_t)2 * BA_RB_IN * 2);
    s.ordr = take((size_t)BA_SBR * 2 * BA_NT * 2);         // per round and list: the round's nodes by class
    s.seg = take((size_t)BA_SBR * 2 * (BA_NCLS + 1) * 2);
    s.order = take((size_t)2 * BA_IN_SB * 2);              // merged: bucket-major node ids of the super-batch
    s.gstart = take((size_t)(BA_IN_NBKT + 1) * 2);
    s.wcnt = take((size_t)(BA_NT / 32) * BA_NCLS * 2);
    s.batch = take((size_t)BA_IN_MAXB * 4);
    s.csr_off = take(((size_t)(1 << m) + 1) * 2);
    (void)ncsr;                                            // the CSR indices are read from global memory (L2)
    s.sub = take(32 * 4);
    s.red = take(64 * 8);
    s.kcw = take(2 * (BA_NMAX_I + 1) * 8);
    s.item = take(16);
    s.total = o;
    return s;
}

// z = b.t from the list b and code(t)
__device__ __forceinline__ uint32_t ba_z_of_tail(uint32_t b, uint32_t tc) {
    const int lt = ba_len_of_code(tc);
    return (1u << (lt + 1)) | (b << lt) | (tc - (1u << lt));
}

template <int MODE>
__global__ void __launch_bounds__(BA_NT, 1) k_enum_in(const __grid_constant__ InArgs a) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int m = a.kc.m, h = a.kc.h, nv = 1 << m;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const InSmem L = enum_in_smem(m, a.ncsr, a.nri);
    const uint32_t ROWD = 1u << m, ROWB = ROWD * 8u;        // half row: operands of the z = b.t, by code(t)

    NodeRec *s_rec = (NodeRec *)(smem + L.rec);
    double *s_ceps = (double *)(smem + L.ceps);
    double *s_rows = (double *)(smem + L.rows);
    double *s_acc = s_rows;                                 // epilogue only
    uint4 *s_bal = (uint4 *)(smem + L.bal);
    uint16_t *s_bnode = (uint16_t *)(smem + L.bnode);
    uint16_t *s_ordr = (uint16_t *)(smem + L.ordr);
    uint16_t *s_seg = (uint16_t *)(smem + L.seg);
    uint16_t *s_order = (uint16_t *)(smem + L.order);
    uint16_t *s_gstart = (uint16_t *)(smem + L.gstart);
    uint16_t *s_wcnt = (uint16_t *)(smem + L.wcnt);
    uint32_t *s_batch = (uint32_t *)(smem + L.batch);
    double *s_rsum = (double *)(smem + L.rsum);
    uint16_t *s_csr_off = (uint16_t *)(smem + L.csr_off);
    uint32_t *s_sub = (uint32_t *)(smem + L.sub);
    double *s_red = (double *)(smem + L.red);
    double *s_w = (double *)(smem + L.kcw);
    double *s_lebar = s_w + (BA_NMAX_I + 1);
    uint32_t *s_item = (uint32_t *)(smem + L.item);        // [0] item, [1] number of batches

    for (int i = tid; i <= nv; i += BA_NT) s_csr_off[i] = a.csr_off[i];
    for (int i = tid; i <= BA_NMAX_I; i += BA_NT) { s_w[i] = a.kc.w[i]; s_lebar[i] = a.kc.lebar[i]; }
    for (int i = tid; i < 2 * BA_RB_IN; i += BA_NT) s_rows[(size_t)i * ROWD] = 0.0;   // position 0: padding pairs

    // which of this warp's chunk slots hold pairs at all (static)
    uint32_t whas = 0;
#pragma unroll
    for (int s = 0; s < 2 * BA_NC; s++)
        if (__any_sync(0xffffffffu, a.owner[(size_t)s * BA_NT + tid] != 0xffffu)) whas |= 1u << s;
    const uint32_t sRows = ba_smem_addr(s_rows);
    const int ev = tid & (nv - 1);                          // v of this thread's empty-z pairs
    const int esub = tid >> m, epn = BA_NT >> m;            // it serves nodes esub, esub + epn, ...
    const int st_pc = tid & ((nv >> 1) - 1), st_i0 = tid >> (m - 1), st_step = BA_NT >> (m - 1);   // staging role
    const int st_lt = st_pc ? ba_len_of_code(2u * (uint32_t)st_pc) : 0;
    const uint32_t st_tv = st_pc ? (2u * (uint32_t)st_pc - (1u << st_lt)) : 0u, st_dst = ba_swz(2u * (uint32_t)st_pc) * 8u;
    __syncthreads();

    unsigned long long cnt_terms = 0, cnt_emb = 0;

    for (;;) {
        if (tid == 0) s_item[0] = (MODE == IN_DEBUG) ? (a.dbg_x >> m) : atomicAdd(a.counter, 1u);
        __syncthreads();
        const uint32_t u = s_item[0];
        if (h < 32 && (u >> (h - a.sym)) != 0) break;
        if (MODE == IN_DEBUG && blockIdx.x != 0) break;

        // ---- Sub[pos] = number of trie nodes below a node whose leftmost embedding ends at pos -------
        if (tid == 0) {
            s_sub[h] = 1u;
            for (int pos = h - 1; pos >= 0; pos--) {
                const int n0 = ba_nextpos(u, h, pos, 0u), n1 = ba_nextpos(u, h, pos, 1u);
                s_sub[pos] = 1u + (n0 < h ? s_sub[n0 + 1] : 0u) + (n1 < h ? s_sub[n1 + 1] : 0u);
            }
        }
        __syncthreads();
        const uint32_t NN = s_sub[0];
        const uint32_t ur = (h > 0) ? (__brev(u) >> (32 - h)) : 0u;      // bit i = symbol at position i

        double acc[2][BA_NC];
#pragma unroll
        for (int b = 0; b < 2; b++)
#pragma unroll
            for (int c = 0; c < BA_NC; c++) acc[b][c] = 0.0;
        double acc_eps = 0.0, acc_rid = 0.0;

        for (uint32_t base = 0; base < NN; base += BA_IN_SB) {
            __syncthreads();                                   // previous super-batch fully consumed
            const int nsb = (NN - base < (uint32_t)BA_IN_SB) ? (int)(NN - base) : BA_IN_SB;
            const int nrounds = (nsb + BA_NT - 1) / BA_NT;
            for (int rd = 0; rd < nrounds; rd++) {
                // ================= phase A: unrank node base + rd*BA_NT + tid, DP along the descent =================
                int key0 = -1, key1 = -1;
                const int nn = (nsb - rd * BA_NT < BA_NT) ? (nsb - rd * BA_NT) : BA_NT;
                if (tid < nn) {
                    uint32_t r = base + (uint32_t)(rd * BA_NT + tid);
                    uint32_t E[BA_HMAX + 1];
#pragma unroll
                    for (int i = 0; i <= BA_HMAX; i++) E[i] = 1u;            // emb(empty, u[0:i]) = 1
                    uint32_t al[9];
                    al[0] = 1u;
#pragma unroll
                    for (int s = 1; s < 9; s++) al[s] = 0u;
                    int pos = 0, k = 0;
                    uint32_t cy = 1u;
                    while (r > 0) {
                        r--;
                        const int n0 = ba_nextpos(u, h, pos, 0u);
                        const uint32_t s0 = (n0 < h) ? s_sub[n0 + 1] : 0u;
                        uint32_t b;
                        int p;
                        if (r < s0) { b = 0u; p = n0; } else { r -= s0; b = 1u; p = ba_nextpos(u, h, pos, 1u); }
                        const uint32_t mm = (b ? ur : ~ur) & ((h >= 32) ? 0xffffffffu : ((1u << h) - 1u));
                        uint32_t run = 0u;
#pragma unroll
                        for (int i = 0; i <= BA_HMAX; i++) {       // N[i] = sum_{j<i, u_j=b} E[j]
                            const uint32_t old = E[i];
                            E[i] = run;
                            if ((mm >> i) & 1u) run += old;
                        }
#pragma unroll
                        for (int s = 8; s >= 1; s--) al[s] = al[s - 1];
                        al[0] = run;                               // emb(y'.b, u)
                        pos = p + 1; k++;
                        cy = (cy << 1) | b;
                    }
                    uint32_t miss0 = ba_nextpos(u, h, pos, 0u) >= h, miss1 = ba_nextpos(u, h, pos, 1u) >= h;
                    // exact channel BDC_{n,klen}: y = y'.z has weight only if |y'| + |z| = klen, 1 <= |z| <= m
                    if ((MODE == IN_SWEEP || MODE == IN_HC) && a.kc.klen >= 0 && !(k < a.kc.klen && a.kc.klen <= k + m)) miss0 = miss1 = 0u;
                    NodeRec rc;
#pragma unroll
                    for (int s = 0; s < 9; s++) rc.a[s] = al[s];
                    rc.id = cy;
                    rc.info = miss0 | (miss1 << 1) | ((uint32_t)(k < 8 ? k : 8) << 8) | ((uint32_t)k << 16);
                    rc.pad = 0u;
                    s_rec[rd * BA_NT + tid] = rc;
                    if (MODE == IN_SWEEP) s_ceps[tid] = a.c[cy];
                    if (miss0) key0 = (int)(cy & (BA_NCLS - 1));
                    if (miss1) key1 = (int)(cy & (BA_NCLS - 1));
                }
                // ================= sort: per list, the round's nodes by class (stable) =================
                ba_bucket_sort<BA_NCLS>(key0, s_ordr + (size_t)(rd * 2 + 0) * BA_NT, s_wcnt, s_seg + (rd * 2 + 0) * (BA_NCLS + 1));
                ba_bucket_sort<BA_NCLS>(key1, s_ordr + (size_t)(rd * 2 + 1) * BA_NT, s_wcnt, s_seg + (rd * 2 + 1) * (BA_NCLS + 1));

                // ================= eps: the pair (v, empty) of every node of the round =================
                auto eps_one = [&](int i) {
                    const NodeRec &rc = s_rec[rd * BA_NT + i];
                    const uint4 r0 = *(const uint4 *)&rc.a[0], r1 = *(const uint4 *)&rc.a[4], r2 = *(const uint4 *)&rc.a[8];
                    const uint32_t cy = r2.y;
                    const int k = (int)(r2.z >> 16);
                    const uint2 e8 = __ldg(a.EPS8 + (size_t)(cy & 255u) * nv + ev);   // alpha_s = 0 beyond k
                    const uint32_t emb = r0.x + r0.y * __byte_perm(e8.x, 0u, 0x4440) + r0.z * __byte_perm(e8.x, 0u, 0x4441) +
                                         r0.w * __byte_perm(e8.x, 0u, 0x4442) + r1.x * __byte_perm(e8.x, 0u, 0x4443) +
                                         r1.y * __byte_perm(e8.y, 0u, 0x4440) + r1.z * __byte_perm(e8.y, 0u, 0x4441) +
                                         r1.w * __byte_perm(e8.y, 0u, 0x4442) + r2.x * __byte_perm(e8.y, 0u, 0x4443);
                    if (MODE == IN_SWEEP) {
                        acc_eps = fma(ba_u2d(emb), s_ceps[i], acc_eps);
                    } else if (MODE == IN_HC) {
                        const double wk = s_w[k];
                        if (wk != 0.0 && emb > 1u) acc_eps = fma(wk * (double)emb, log2((double)emb) - s_lebar[k], acc_eps);
                        else if (wk != 0.0) acc_eps = fma(wk, -s_lebar[k], acc_eps);
                    } else if (MODE == IN_DEBUG) {
                        if (((u << m) | (uint32_t)ev) == a.dbg_x) a.dbg_out[cy - 1u] = emb;
                    } else {
                        cnt_terms += 1ull; cnt_emb += emb;
                    }
                };
                if ((MODE == IN_SWEEP || MODE == IN_HC) && a.kc.klen >= 0) {      // exact channel: only |y'| = klen has weight
                    for (int i = esub; i < nn; i += epn)
                        if ((int)(s_rec[rd * BA_NT + i].info >> 16) == a.kc.klen) eps_one(i);
                } else {
#pragma unroll 8
                    for (int i = esub; i < nn; i += epn) eps_one(i);
                }
                __syncthreads();                               // s_ceps is rewritten by the next round
            }
            // ================= merge the rounds: bucket (b, cls) = its runs in round order =================
            if (tid < 32) {
                int cnt = 0;
                const int bq = tid >> 4, cq = tid & (BA_NCLS - 1);          // BA_IN_NBKT = 32 buckets, one per lane
                for (int rd = 0; rd < nrounds; rd++) {
                    const uint16_t *sg = s_seg + (rd * 2 + bq) * (BA_NCLS + 1) + cq;
                    cnt += sg[1] - sg[0];
                }
                int incl = cnt;
                for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
                int pos = incl - cnt;
                s_gstart[tid] = (uint16_t)pos;
                if (tid == 31) s_gstart[32] = (uint16_t)incl;
                for (int rd = 0; rd < nrounds; rd++) {
                    const uint16_t *sg = s_seg + (rd * 2 + bq) * (BA_NCLS + 1) + cq;
                    const uint16_t *od = s_ordr + (size_t)(rd * 2 + bq) * BA_NT;
                    for (int i = sg[0]; i < sg[1]; i++) s_order[pos++] = (uint16_t)(rd * BA_NT + od[i]);
                }
                __syncwarp();
                if (tid == 0) {                                // batches: <= BA_RB_IN consecutive nodes of one bucket
                    int nb = 0;
                    for (int kq = 0; kq < BA_IN_NBKT; kq++)
                        for (int off = s_gstart[kq]; off < s_gstart[kq + 1]; off += BA_RB_IN) {
                            const int len = (s_gstart[kq + 1] - off < BA_RB_IN) ? (s_gstart[kq + 1] - off) : BA_RB_IN;
                            s_batch[nb++] = (uint32_t)off | ((uint32_t)len << 16) | ((uint32_t)kq << 24);
                        }
                    s_item[1] = (uint32_t)nb;
                }
            }
            __syncthreads();

            // ================= phase B: batches of one (list, class) =================
            const int nbatch = (int)s_item[1];
            auto stage = [&](int j) {                          // half rows, alpha_0..3 and node ids of batch j
                const uint32_t bi = s_batch[j];
                const int start = (int)(bi & 0xffffu), len = (int)((bi >> 16) & 0xffu), buf = j & 1;
                const uint32_t b = (bi >> 24) / BA_NCLS;
                if (MODE == IN_SWEEP) {
                    // 16-byte pieces (positions 2pc, 2pc+1), 2^{m-1} per half row: a thread always copies the same
                    // piece, of every st_step-th row
                    for (int i = st_i0; i < len; i += st_step) {
                        const uint32_t cy = s_rec[s_order[start + i]].id;
                        const uint32_t dst = sRows + ((uint32_t)(buf * BA_RB_IN + i) * ROWD) * 8u;
                        if (st_pc == 0)                        // position 1: t empty, z = "b"
                            ba_cp_async8(dst + 8u, a.c + ((cy << 1) + b));             // codes fit 32 bits (n <= 30)
                        else
                            ba_cp_async16(dst + st_dst, a.c + ((cy << (st_lt + 1)) + (b << st_lt) + st_tv));
                    }
                }
                if (tid < len) {
                    const int node = s_order[start + tid];
                    s_bal[buf * BA_RB_IN + tid] = *(const uint4 *)&s_rec[node].a[0];
                    s_bnode[buf * BA_RB_IN + tid] = (uint16_t)node;
                }
            };
            auto flush = [&](int j) {                          // thread v collects the rider sums of batch j
                if (MODE != IN_SWEEP && MODE != IN_HC) return;
                if (tid >= nv) return;
                const int kq = (int)(s_batch[j] >> 24), buf = j & 1;
                const uint16_t *cs = a.ri_csr + (size_t)((kq % BA_NCLS) * 2 + kq / BA_NCLS) * (nv + 1) + tid;
                const int e0 = cs[0], e1 = cs[1];
                for (int e = e0; e < e1; e++) acc_rid += s_rsum[((size_t)buf * 2) * a.nri + e] + s_rsum[((size_t)buf * 2 + 1) * a.nri + e];
            };
            if (nbatch > 0) stage(0);
            for (int j = 0; j < nbatch; j++) {
                const uint32_t bi = s_batch[j];
                const int len = (int)((bi >> 16) & 0xffu), kq = (int)(bi >> 24), buf = j & 1;
                const int cls = kq % BA_NCLS, bsel = kq / BA_NCLS;
                // the pairs of a chunk do not depend on the staged rows: fetch slot 0 before waiting, and slot c+1
                // while slot c is being computed, so that one L2 latency per batch is exposed at most
                const uint2 *F = a.FI + (((size_t)cls * 2 + bsel) * BA_NC) * BA_C * BA_NT + tid;
                uint32_t nbp[BA_C], nad[BA_C];
#pragma unroll
                for (int q = 0; q < BA_C; q++) { const uint2 pr = __ldg(F + (size_t)q * BA_NT); nbp[q] = pr.x; nad[q] = pr.y; }
                ba_cp_async_wait_all();
                __syncthreads();                               // batch j staged; batch j-1 fully consumed
                if (j + 1 < nbatch) stage(j + 1);
                if (j > 0) flush(j - 1);
                const uint32_t rowbase = sRows + (uint32_t)(buf * BA_RB_IN) * ROWB;
                const uint4 *bal = s_bal + buf * BA_RB_IN;
                const uint16_t *bnode = s_bnode + buf * BA_RB_IN;
#pragma unroll
                for (int b = 0; b < 2; b++) {
                    if (b != bsel) continue;
                    // ---- fast pairs -----------------------------------------------------------------------
#pragma unroll
                    for (int c = 0; c < BA_NC; c++) {
                        uint32_t bp[BA_C], ad[BA_C];
#pragma unroll
                        for (int q = 0; q < BA_C; q++) { bp[q] = nbp[q]; ad[q] = nad[q]; }
                        if (c + 1 < BA_NC) {
#pragma unroll
                            for (int q = 0; q < BA_C; q++) {
                                const uint2 pr = __ldg(F + (size_t)((c + 1) * BA_C + q) * BA_NT);
                                nbp[q] = pr.x; nad[q] = pr.y;
                            }
                        }
                        if (!((whas >> (b * BA_NC + c)) & 1u)) continue;
                        if (MODE == IN_SWEEP) {
                            acc[b][c] = ba_fast_chunk(acc[b][c], bal, rowbase, ROWB, len, bp, ad);
                        } else {
                            const uint32_t ov = a.owner[((size_t)b * BA_NC + c) * BA_NT + tid];
                            for (int i = 0; i < len; i++) {
                                const uint4 al = bal[i];
                                const NodeRec &rc = s_rec[bnode[i]];
                                const int k = (int)(rc.info >> 16);
#pragma unroll
                                for (int q = 0; q < BA_C; q++) {
                                    if (!(bp[q] & 0xffu)) continue;
                                    const uint32_t emb = al.x * (bp[q] & 0xffu) + al.y * ((bp[q] >> 8) & 0xffu) +
                                                         al.z * ((bp[q] >> 16) & 0xffu) + al.w * (bp[q] >> 24);
                                    const uint32_t cz = ba_z_of_tail((uint32_t)b, ba_swz(ad[q] >> 3));
                                    const int jz = ba_len_of_code(cz);
                                    if (MODE == IN_HC) {
                                        const double wk = s_w[k + jz];
                                        if (wk != 0.0) {
                                            const double le = (emb > 1u) ? log2((double)emb) : 0.0;
                                            acc[b][c] = fma(wk * (double)emb, le - s_lebar[k + jz], acc[b][c]);
                                        }
                                    } else if (MODE == IN_DEBUG) {
                                        if (((u << m) | ov) == a.dbg_x)
                                            a.dbg_out[((size_t)rc.id << jz) + (cz - (1u << jz)) - 1u] = emb;
                                    } else {
                                        cnt_terms += 1ull; cnt_emb += emb;
                                    }
                                }
                            }
                        }
                    }
                    // ---- riders: deep pairs of this class, one per thread ------------------------------------
                    const int nr = a.ri_cnt[cls * 2 + b];
                    // two replicas of the rider set (threads 255 - e and 511 - e), each takes every other node
                    const int re = (BA_NT / 2 - 1) - (tid & (BA_NT / 2 - 1)), rh = tid / (BA_NT / 2);
                    if ((BA_NT / 2) - 32 * ((warp & (BA_NT / 64 - 1)) + 1) < nr) {
                        double s = 0.0;
                        if (re < nr) {
                            const uint4 rd = __ldg(a.RI + ((size_t)cls * 2 + b) * a.nri + re);
                            const uint32_t B0 = rd.x & 0xffu, B1 = (rd.x >> 8) & 0xffu, B2 = (rd.x >> 16) & 0xffu, B3 = rd.x >> 24;
                            const uint32_t B4 = rd.y & 0xffu, ov = rd.y >> 16;
                            const uint32_t cz = ba_z_of_tail((uint32_t)b, ba_swz(rd.z >> 3));
                            const int jz = ba_len_of_code(cz);
                            const uint32_t *r8 = a.RI8 + ((size_t)cls * 2 + b) * 16 * a.nri + re;
#pragma unroll 4                                           // four independent L2 reads of the chain tails in flight
                            for (int i = rh; i < len; i += 2) {
                                const NodeRec &rc = s_rec[bnode[i]];
                                const uint4 r0 = *(const uint4 *)&rc.a[0], r1 = *(const uint4 *)&rc.a[4], r2 = *(const uint4 *)&rc.a[8];
                                const uint32_t cy = r2.y;
                                const int k = (int)(r2.z >> 16);
                                const uint32_t x8 = __ldg(r8 + (size_t)((cy >> 4) & 15u) * a.nri);   // alpha_s = 0 beyond k
                                const uint32_t emb = r0.x * B0 + r0.y * B1 + r0.z * B2 + r0.w * B3 + r1.x * B4 +
                                                     r1.y * __byte_perm(x8, 0u, 0x4440) + r1.z * __byte_perm(x8, 0u, 0x4441) +
                                                     r1.w * __byte_perm(x8, 0u, 0x4442) + r2.x * __byte_perm(x8, 0u, 0x4443);
                                if (MODE == IN_SWEEP) {
                                    s = fma(ba_u2d(emb), ba_lds_f64(rowbase + (uint32_t)i * ROWB + rd.z), s);
                                } else if (MODE == IN_HC) {
                                    const double wk = s_w[k + jz];
                                    if (wk != 0.0) {
                                        const double le = (emb > 1u) ? log2((double)emb) : 0.0;
                                        s = fma(wk * (double)emb, le - s_lebar[k + jz], s);
                                    }
                                } else if (MODE == IN_DEBUG) {
                                    if (((u << m) | ov) == a.dbg_x) a.dbg_out[((size_t)cy << jz) + (cz - (1u << jz)) - 1u] = emb;
                                } else {
                                    cnt_terms += 1ull; cnt_emb += emb;
                                }
                            }
                        }
                        if ((MODE == IN_SWEEP || MODE == IN_HC) && re < nr) s_rsum[((size_t)buf * 2 + rh) * a.nri + re] = s;
                    }
                }
            }
            if (nbatch > 0) {
                __syncthreads();                               // rider sums of the last batch are visible
                flush(nbatch - 1);
            }
        }

        // ---- epilogue: thread v owns x = u.v ------------------------------------------------------------
        __syncthreads();                                       // all rows consumed: the staging area becomes s_acc
        if (MODE == IN_SWEEP || MODE == IN_HC) {
#pragma unroll
            for (int b = 0; b < 2; b++)
#pragma unroll
                for (int c = 0; c < BA_NC; c++) s_acc[((size_t)b * BA_NC + c) * BA_NT + tid] = acc[b][c];
            s_acc[(size_t)2 * BA_NC * BA_NT + tid] = acc_eps;
            __syncthreads();
            double r0 = 0.0, r1 = -INFINITY, r2 = 0.0;
            if (tid < nv) {
                double S = acc_rid;
                for (int t = ev; t < BA_NT; t += nv) S += s_acc[(size_t)2 * BA_NC * BA_NT + t];
                for (int q = s_csr_off[tid]; q < s_csr_off[tid + 1]; q++) S += s_acc[__ldg(a.csr_idx + q)];
                const size_t x = ((size_t)u << m) | (size_t)tid;
                const size_t xc = (((size_t)1 << a.kc.n) - 1) - x;     // complement: same row of emb up to cpl
                if (MODE == IN_HC) {
                    a.Hc[x] = S;
                    if (a.sym) a.Hc[xc] = S;
                } else {
                    const double Dx = a.Hc[x] - S;
                    a.D[x] = Dx;
                    const double px = a.p[x];
                    r0 = px * Dx; r1 = Dx; r2 = px * exp2(Dx);
                    if (a.sym) { a.D[xc] = Dx; r0 += r0; r2 += r2; }  // p(xc) = p(x) bit for bit (checked on the host)
                }
            }
            if (MODE == IN_SWEEP) {
                for (int o = 16; o > 0; o >>= 1) {
                    r0 += __shfl_xor_sync(0xffffffffu, r0, o);
                    r1 = fmax(r1, __shfl_xor_sync(0xffffffffu, r1, o));
                    r2 += __shfl_xor_sync(0xffffffffu, r2, o);
                }
                if (lane == 0) { s_red[warp * 3] = r0; s_red[warp * 3 + 1] = r1; s_red[warp * 3 + 2] = r2; }
                __syncthreads();
                if (tid == 0) {
                    double t0 = 0.0, t1 = -INFINITY, t2 = 0.0;
                    for (int w = 0; w < BA_NT / 32; w++) {
                        t0 += s_red[w * 3];
                        t1 = fmax(t1, s_red[w * 3 + 1]);
                        t2 += s_red[w * 3 + 2];
                    }
                    a.part[(size_t)u * 3] = t0;
                    a.part[(size_t)u * 3 + 1] = t1;
                    a.part[(size_t)u * 3 + 2] = t2;
                }
            }
            __syncthreads();
            for (int i = tid; i < 2 * BA_RB_IN; i += BA_NT) s_rows[(size_t)i * ROWD] = 0.0;   // restore position 0 of the rows
        }
        if (MODE == IN_DEBUG) break;
        __syncthreads();
    }
    if (MODE == IN_COUNT) {
        atomicAdd(&a.cnt[0], cnt_terms);
        atomicAdd(&a.cnt[1], cnt_emb);
    }
}
