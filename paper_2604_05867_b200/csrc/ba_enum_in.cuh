// ba_enum_in.cuh -- input sweep: for every x, enumerate its distinct subsequences y
// with their integer embedding counts emb(y,x) exactly once each.
//
// Work item = (high part u of h bits, list b) with the 2^m inputs x = u.v; one persistent CTA per SM takes
// items from an atomic counter.  Item (u, b) visits the terms y = y'.z with z[0] = b and, for b = 0, the terms
// y = y' (z empty).  Per item, in super-batches of BA_SBR * BA_NT nodes:
//   phase A  (BA_SBR rounds) every thread UNRANKS one node per round: the r-th distinct subsequence y' of
//            u in trie pre-order (the paper's stringUnrank idea, Alg. 4, with the subtree sizes
//            Sub[pos] in the role of the Count table P:260-274 and NextPos P:256-258 done with clz on bit
//            masks), and carries the integer embedding-count DP  E[i] = emb(y', u[0:i])  in registers
//            along the descent; the node record {alpha_0..8, code(y'), mask} goes to shared memory.
//   sort     the nodes that carry list b (b cannot follow y' in u) are ranked, stably, by class; the rounds' runs are
//            merged into one order.
//   phase B  batches of <= BA_RB_IN nodes of one class.  The operands c(y'.z), z = b.t, of a node
//            form a HALF ROW of 2^m doubles indexed by code(t): one row of crow, staged by warp 0 with one bulk copy,
//            double buffered; FULL / EMPTY mbarriers are the only per-batch synchronisation.  Every thread owns BA_KG
//            groups of BA_GP pairs (ba_internal.h "GROUPS"): a group is one z with up to 4 different v, so c(y'.z) is read once per node and group; the
//            slots' B_0..B_3 are constants of the batch, and the loop over the nodes of the batch costs, per (x,y) term,
//                 1-2 IDP.2A (emb) + 1 exact u32->f64 + 1 DFMA
//            with one FP64 accumulator per slot kept in a register for the whole item.  Deep pairs
//            ride along, one per thread, their partial sums handed to thread v through shared memory
//            in a fixed order.
//   (v, empty) IN_SWEEP sums these pairs in factored form: G sums per suffix of y', expanded once per item (P:181 at
//            the tile boundary; see "G sums" below and DESIGN.md section 5); the other modes enumerate them.
//   epilogue thread v adds the accumulators of v's slots in a fixed order: S_b(x) = sum_{y in item} emb(y,x) c(y).
// k_in_final (ba_stream.cuh) forms D(x) = Hc(x) - S_0(x) - S_1(x) and the first stage of the reductions of 8(a3).
// MODE:
//   IN_SWEEP  S_b(x)
//   IN_HC     H_b(x) = sum_{y in item} w_k (emb log2(emb) - emb log2(ebar_k))   (iteration independent; built once per ctx;
//             centred term by term: the partial sums stay of the size of D)
//   IN_DEBUG  emb_out[idx(y)] = emb(y,x) for one x     (ba_debug_emb_row; two CTAs, one per list)
//   IN_COUNT  number of visited terms and sum of emb   (ba_debug_count_terms)
#pragma once
#include "ba_internal.h"

enum { IN_SWEEP = 0, IN_HC = 1, IN_DEBUG = 2, IN_COUNT = 3 };

#define BA_ELOG_S 16384                                    // head of the e log2(e) table kept in shared memory (IN_HC): it takes the
                                                           // place of the operand rows, which that pass does not stage
#define BA_IN_SB (BA_SBR * BA_NT)                           // nodes per super-batch
#define BA_IN_NBKT (2 * BA_NCLS)                            // buckets: class, with / without list b (the latter: b = 0 only)
#define BA_IN_MAXB (BA_IN_NBKT + BA_IN_SB / BA_RB_IN)
#define BA_IN_NG (512 + 5 * BA_NCLS)                        // G sums of an item: by code(w), |w| >= 5; by (class, s), s <= 4

struct InArgs {
    KConst kc;
    GroupDev g;               // schedule of the input sweep (owner = v, operand position = code(z[1:]))
    const uint2 *EPS8;        // [256][2^m]: B(sigma_s, v), s = 0..7, of the pair (v, empty)
    const uint32_t *EPSH;     // [cls][8][2^m]: B_4..B_7 of the pair (v, empty) by the sigma bits 4..6: a class's slice
    const double *c;          // IN_SWEEP: c[code(y)], 2^{n+1} entries (entry 0 unused)
    const double *crow;       // IN_SWEEP: the same by rows (code(y'), b) of 2^m operands (k_out_final)
    const uint32_t *LTV_off;  // [2^m + 1]: the subsequences w of v ...
    const uint32_t *LTV;      // ... as code(w) << 8 | emb(w, v)   (IN_SWEEP: the pairs (v, empty) in factored form)
    const double *elog;       // IN_HC: elog[e] = e log2(e), e < BA_ELOG_N
    double *S;                // out: [2][2^n] partial sums of the two lists (IN_SWEEP: S_b, IN_HC: H_b)
    double *park;             // [grid][2][BA_NSLOT][BA_NT]: the accumulators of the schedule that is not running
    unsigned int *counter;    // work counter (zeroed before launch)
    int sym;                  // 1: p(x) = p(~x) (Theorem 4): only the u with leading bit 0 are enumerated
    uint32_t dbg_x;           // IN_DEBUG
    uint32_t *dbg_out;        // IN_DEBUG: NY zero-filled
    unsigned long long *cnt;  // IN_COUNT: [0] terms, [1] emb sum
};

struct InSmem { size_t rec, slice, rslice, rows, mbar, bal, ordr, seg, order, skey, g2map, gstart, wcnt, batch, rsum, sub, kcw, item, total; };

// sweep = the layout of IN_SWEEP (no riders: nr counts the deep-part targets; sorted keys and split maps instead of the
// rider slices); otherwise the layout of the modes that enumerate every term (riders, nr = capacity of the rider set)
__host__ __device__ static inline InSmem enum_in_smem(int nr, bool sweep) {
    if (sweep) nr = BA_G2_NT;
    InSmem s;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 15) & ~(size_t)15; return at; };
    s.rec = take((size_t)BA_IN_SB * sizeof(NodeRec));
    s.rsum = take((size_t)4 * 2 * nr * 8 > (size_t)BA_NT * 8 ? (size_t)4 * 2 * nr * 8 : (size_t)BA_NT * 8);   // rider sums of a batch, two replicas,
                                                           // four batches deep (collected two batches late); the epilogue parks acc_eps there
    s.slice = take((size_t)2 * 8 * ((size_t)1 << BA_MLOW) * 4);    // B_4..B_7 of the pairs (v, empty) of a class, double buffered
    s.rslice = take(sweep ? 0 : (size_t)2 * 8 * nr * 4);   // B_4..B_7 of the riders of a class, double buffered
    size_t rows = (size_t)2 * BA_RB_IN * BA_ROWB, ac = (size_t)2 * BA_NSLOT * BA_NT * 8;   // both schedules' accumulators
    s.rows = take(rows > ac ? rows : ac);                  // the epilogue's accumulator staging aliases the rows
    s.mbar = take(4 * 8);                                  // FULL and EMPTY barriers of the two row buffers
    s.bal = take((size_t)2 * BA_RB_IN * sizeof(BalRec));
    s.ordr = take((size_t)BA_SBR * BA_NT * 2);             // per round: the round's nodes by class
    s.seg = take((size_t)BA_SBR * (BA_IN_NBKT + 1) * 2);
    s.order = take((size_t)BA_IN_SB * 2);                  // merged: class-major node ids of the super-batch
    s.skey = take(sweep ? (size_t)BA_IN_SB * 2 : 0);                 // in the same order: last 8 symbols of y' | min(|y'|, 15) << 8 (G sums)
    s.g2map = take(sweep ? (size_t)2 * 480 * 8 : 0);                 // per list and owner thread of w: (class, target) of the splits of w (deep part)
    s.gstart = take((size_t)(BA_IN_NBKT + 1) * 2);
    s.wcnt = take((size_t)(BA_NT / 32) * BA_IN_NBKT * 2);
    s.batch = take((size_t)BA_IN_MAXB * 4);
    s.sub = take(32 * 4);
    s.kcw = take(2 * (BA_NMAX_I + 1) * 8);
    s.item = take(16);
    s.total = o;
    return s;
}

#define BA_ELOG_N 65536
// e log2(e) of an embedding count: a table for the (overwhelmingly many) small counts, the library log2 otherwise
__device__ __forceinline__ double ba_elog2e(uint32_t e, const double *tab, const double *stab) {
    if (e < BA_ELOG_S) return stab[e];
    if (e < BA_ELOG_N) return __ldg(tab + e);
    return (double)e * log2((double)e);
}

// z = b.t from the list b and the position of its operand in the staged half row: code(t), except that the
// one-symbol z = "b" (t empty) sits at position b
__device__ __forceinline__ uint32_t ba_z_of_tail(uint32_t b, uint32_t pos) {
    const uint32_t tc = (pos < 2u) ? 1u : pos;
    const int lt = ba_len_of_code(tc);
    return (1u << (lt + 1)) | (b << lt) | (tc - (1u << lt));
}

template <int MODE>
__global__ void __launch_bounds__(BA_NT, 1) k_enum_in(const __grid_constant__ InArgs a) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int m = a.kc.m, h = a.kc.h, nv = 1 << m;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const InSmem L = enum_in_smem(a.g.nr, MODE == IN_SWEEP);

    NodeRec *s_rec = (NodeRec *)(smem + L.rec);
    uint32_t *s_slice = (uint32_t *)(smem + L.slice);
    uint32_t *s_rslice = (uint32_t *)(smem + L.rslice);
    // IN_SWEEP forms the pairs (v, empty) in factored form (see "G sums" below) and stages no slice of them: their area
    // holds c(y') of the super-batch's nodes and the G sums of the item
    double *s_c = (double *)s_slice;
    double *s_G = s_c + BA_IN_SB;
    static_assert((size_t)(BA_IN_SB + BA_IN_NG) * 8 <= (size_t)2 * 8 * ((size_t)1 << BA_MLOW) * 4, "c(y') and the G sums live in the slice area");
    double *s_rows = (double *)(smem + L.rows);
    double *s_acc = s_rows;                                 // epilogue only
    double *s_elog = s_rows;                                // IN_HC: the table's head; the epilogue overwrites it, so it is
    auto load_elog = [&]() {                                // fetched again (128 KB from L2) after every item
        static_assert((size_t)BA_ELOG_S * 8 <= (size_t)2 * BA_RB_IN * BA_ROWB, "the table head lives in the row buffers");
        for (int i = tid; i < BA_ELOG_S / 2; i += BA_NT) ((double2 *)s_elog)[i] = __ldg((const double2 *)a.elog + i);
    };
    BalRec *s_bal = (BalRec *)(smem + L.bal);
    uint16_t *s_ordr = (uint16_t *)(smem + L.ordr);
    uint16_t *s_seg = (uint16_t *)(smem + L.seg);
    uint16_t *s_order = (uint16_t *)(smem + L.order);
    uint16_t *s_skey = (uint16_t *)(smem + L.skey);
    uint2 *s_g2map = (uint2 *)(smem + L.g2map);
    if (MODE == IN_SWEEP && tid < 480) {                    // g2map: see "deep part" below; static but for the list
        const uint32_t code = 32u + (uint32_t)tid;
        const int Lw = ba_len_of_code(code);
        const uint32_t wv = code - (1u << Lw);
        for (int bb = 0; bb < 2; bb++) {
            uint32_t gm[2] = {0u, 0u};
            if (Lw <= m && m >= 5)
                for (int s = 4; s < Lw && s < 8; s++) {
                    const int zl = Lw - s;
                    const uint32_t z = wv & ((1u << zl) - 1u), sig = wv >> zl;
                    if ((int)((z >> (zl - 1)) & 1u) != bb) continue;
                    const uint32_t tc = (1u << (zl - 1)) | (z & ((1u << (zl - 1)) - 1u)), ext = sig >> 4;
                    const uint32_t t = (s == 4) ? tc - 1u : (s == 5) ? 15u + ext * 7u + tc - 1u : (s == 6) ? 29u + ext * 3u + tc - 1u : 41u + ext;
                    gm[(s - 4) >> 1] |= (0x8000u | ((sig & 15u) << 8) | t) << (16 * ((s - 4) & 1));
                }
            s_g2map[bb * 480 + tid] = make_uint2(gm[0], gm[1]);
        }
    }
    uint16_t *s_gstart = (uint16_t *)(smem + L.gstart);
    uint16_t *s_wcnt = (uint16_t *)(smem + L.wcnt);
    uint32_t *s_batch = (uint32_t *)(smem + L.batch);
    double *s_rsum = (double *)(smem + L.rsum);
    uint32_t *s_sub = (uint32_t *)(smem + L.sub);
    double *s_w = (double *)(smem + L.kcw);
    double *s_lebar = s_w + (BA_NMAX_I + 1);
    uint32_t *s_item = (uint32_t *)(smem + L.item);        // [0] item, [1] number of batches

    for (int i = tid; i <= BA_NMAX_I; i += BA_NT) { s_w[i] = a.kc.w[i]; s_lebar[i] = a.kc.lebar[i]; }
    const uint32_t sFull = ba_smem_addr(smem + L.mbar), sEmpty = sFull + 16u;
    if (tid == 0) {
        ba_mbar_init(sFull, 32u); ba_mbar_init(sFull + 8u, 32u);        // the 32 lanes of the staging warp; copies count in bytes
        ba_mbar_init(sEmpty, BA_NT / 32); ba_mbar_init(sEmpty + 8u, BA_NT / 32);   // one arrival per warp that has left the batch
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (MODE == IN_HC) load_elog();
    else
        for (int i = tid; i < 2 * BA_RB_IN * (int)(BA_ROWB / 8); i += BA_NT) s_rows[i] = 0.0;   // unused slots read finite operands
    uint32_t gb = 0;                                        // batches staged so far by this CTA (uniform): buffer and phase

    const uint32_t sRows = ba_smem_addr(s_rows);
    const int ev = tid & (nv - 1);                          // v of this thread's empty-z pairs
    const int esub = tid >> m, epn = BA_NT >> m;            // it serves nodes esub, esub + epn, ...
    const bool may_big = h > 18;                            // C(h, h/2) >= 2^16 first at h = 19
    __syncthreads();

    unsigned long long cnt_terms = 0, cnt_emb = 0;
    const size_t NX = (size_t)1 << a.kc.n;

    for (;;) {
        if (tid == 0) s_item[0] = (MODE == IN_DEBUG) ? (((a.dbg_x >> m) << 1) | blockIdx.x) : atomicAdd(a.counter, 1u);
        __syncthreads();
        const uint32_t u = s_item[0] >> 1;
        const int b = (int)(s_item[0] & 1u);
        if (h < 31 && (u >> (h - a.sym)) != 0) break;
        if (MODE == IN_DEBUG && blockIdx.x > 1) break;
        const int klen = (MODE == IN_SWEEP || MODE == IN_HC) ? a.kc.klen : -1;
        // The pairs (v, empty) (list 0 serves them).  With the concatenation identity at the tile boundary,
        //     sum_{y' in u} c(y') emb(y', u.v) = sum_w G(w) emb(w, v),   G(w) = sum_{y' ending in w} c(y') alpha_{|w|}(y'),
        // so IN_SWEEP adds c(y') alpha_s of every node to the nine G sums of its suffixes (eps_fact) and expands them
        // once per item; the other modes need every emb on its own and enumerate the 2^m terms of a node (eps_enum).
        const bool eps_fact = MODE == IN_SWEEP && b == 0, eps_enum = MODE != IN_SWEEP && b == 0;
        if (MODE == IN_SWEEP)
            for (int i = tid; i < BA_IN_NG; i += BA_NT) s_G[i] = 0.0;
        // The deep part of the chains (s >= 4), IN_SWEEP: the same identity with z kept,
        //     sum_{y', z} c(y'.z) sum_{s>=4} alpha_s emb(sigma_s.z, v) = sum_w G2(w) emb(w, v),  G2(w) = sum_{sigma_s.z = w} c(y'.z) alpha_s,
        // so every pair keeps a plain slot with B_0..B_3 (schedule `inf`, no riders) and G2 joins the G sums.  Under one
        // class and list there are BA_G2_NT = 49 targets (s, bits 4..s-1 of sigma_s, z): 15 + 2*7 + 4*3 + 8*1; a batch's
        // targets are summed by the last 49 threads of each half of the CTA (every other node each) from the staged
        // rows, and handed through shared memory to the owner thread of w = sigma_s.z, which collects them two batches
        // later (as the rider sums of the other modes).  g2map: the (class, target) of the <= 4 splits of this thread's w.
        double acc_g2 = 0.0;

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

        // ---- per item: the thread's groups (static per list) -----------------------------------------
        // the slots of a thread belong to one of two schedules: sc = last symbol of y' (class bit 0).  The batches
        // of a super-batch run schedule 0 first, then schedule 1; at the switch the accumulators are parked in global
        // memory (L2) and the other schedule's are fetched: twice per super-batch.
        int cur_sc = -1, wmeta = 0;
        uint32_t parked = 0u;                                  // bit sc: schedule sc has accumulators in its parking place
        uint32_t gaddr[BA_KG] = {0u, 0u, 0u, 0u};
        double *park = a.park + (size_t)blockIdx.x * 2 * BA_NSLOT * BA_NT + tid;
        double acc[BA_NSLOT];
#pragma unroll
        for (int s = 0; s < BA_NSLOT; s++) acc[s] = 0.0;
        double acc_eps = 0.0, acc_rid = 0.0;

        for (uint32_t base = 0; base < NN; base += BA_IN_SB) {
            __syncthreads();                                   // previous super-batch fully consumed
            const int nsb = (NN - base < (uint32_t)BA_IN_SB) ? (int)(NN - base) : BA_IN_SB;
            const int nrounds = (nsb + BA_NT - 1) / BA_NT;
            for (int rd = 0; rd < nrounds; rd++) {
                // ================= phase A: unrank node base + rd*BA_NT + tid, DP along the descent =================
                int key = -1;
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
                        uint32_t bb;
                        int p;
                        if (r < s0) { bb = 0u; p = n0; } else { r -= s0; bb = 1u; p = ba_nextpos(u, h, pos, 1u); }
                        const uint32_t mm = (bb ? ur : ~ur) & ((h >= 32) ? 0xffffffffu : ((1u << h) - 1u));
                        uint32_t run = 0u;
#pragma unroll
                        for (int i = 0; i <= 8; i++) {             // N[i] = sum_{j<i, u_j=b} E[j]
                            const uint32_t old = E[i];
                            E[i] = run;
                            if ((mm >> i) & 1u) run += old;
                        }
                        if (h > 8) {                               // mm has no bit at or above h: entries beyond h are never read
#pragma unroll
                            for (int i = 9; i <= 16; i++) {
                                const uint32_t old = E[i];
                                E[i] = run;
                                if ((mm >> i) & 1u) run += old;
                            }
                        }
                        if (h > 16) {
#pragma unroll
                            for (int i = 17; i <= BA_HMAX; i++) {
                                const uint32_t old = E[i];
                                E[i] = run;
                                if ((mm >> i) & 1u) run += old;
                            }
                        }
#pragma unroll
                        for (int s = 8; s >= 1; s--) al[s] = al[s - 1];
                        al[0] = run;                               // emb(y'.b, u)
                        pos = p + 1; k++;
                        cy = (cy << 1) | bb;
                    }
                    uint32_t missb = ba_nextpos(u, h, pos, (uint32_t)b) >= h;
                    // exact channel BDC_{n,klen}: y = y'.z has weight only if |y'| + |z| = klen, 1 <= |z| <= m
                    if (klen >= 0 && !(k < klen && klen <= k + m)) missb = 0u;
                    NodeRec rc;
#pragma unroll
                    for (int s = 0; s < 9; s++) rc.a[s] = al[s];
                    rc.id = cy;
                    rc.info = missb | ((uint32_t)(k < 8 ? k : 8) << 8) | ((uint32_t)k << 16);
                    s_rec[rd * BA_NT + tid] = rc;
                    if (eps_fact) {                                // c(y') of the node (exact channel: only |y'| = klen has weight)
                        if (klen < 0 || k == klen) ba_cp_async8(ba_smem_addr(&s_c[rd * BA_NT + tid]), a.c + cy);
                        else s_c[rd * BA_NT + tid] = 0.0;
                    }
                    // buckets: class for the nodes that carry list b; for b = 0 the others follow in buckets 16 + class:
                    // they contribute the pair (v, empty) only (exact channel: only if |y'| = klen)
                    if (missb) key = (int)(cy & (BA_NCLS - 1));
                    else if (b == 0 && (klen < 0 || k == klen)) key = BA_NCLS + (int)(cy & (BA_NCLS - 1));
                }
                // ================= sort: the round's nodes by bucket (stable) =================
                ba_bucket_sort<BA_IN_NBKT>(key, s_ordr + (size_t)rd * BA_NT, s_wcnt, s_seg + rd * (BA_IN_NBKT + 1));
            }
            // ================= merge the rounds: bucket = its runs in round order =================
            uint16_t *s_roff = s_wcnt;                         // [round][bucket]: where the round's run starts inside the bucket
            if (tid < 32) {
                int cnt = 0;
                for (int rd = 0; rd < nrounds; rd++) {
                    const uint16_t *sg = s_seg + rd * (BA_IN_NBKT + 1) + tid;
                    s_roff[rd * BA_IN_NBKT + tid] = (uint16_t)cnt;
                    cnt += sg[1] - sg[0];
                }
                int incl = cnt;
                for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
                s_gstart[tid] = (uint16_t)(incl - cnt);
                if (tid == 31) s_gstart[32] = (uint16_t)incl;
                // batches: <= BA_RB_IN consecutive nodes of one bucket, class-major (list-carrying bucket, then the other);
                // lane l takes the l-th bucket of that order
                const int cq_l = ((lane >> 1) & 7) * 2 + (lane >> 4);          // class order: bit 0 = 0 first (one schedule switch)
                const int kq = (lane & 1) * BA_NCLS + cq_l;
                const int ck = __shfl_sync(0xffffffffu, cnt, kq), gk = __shfl_sync(0xffffffffu, incl - cnt, kq);
                const int ckb = (MODE == IN_SWEEP && kq >= BA_NCLS) ? 0 : ck;   // IN_SWEEP: no batches without list b
                const int nbk = (ckb + BA_RB_IN - 1) / BA_RB_IN;
                int bincl = nbk;
                for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, bincl, o); if (lane >= o) bincl += t; }
                int nb = bincl - nbk;
                for (int off = 0; off < ckb; off += BA_RB_IN) {
                    const int len = (ckb - off < BA_RB_IN) ? (ckb - off) : BA_RB_IN;
                    s_batch[nb++] = (uint32_t)(gk + off) | ((uint32_t)len << 16) | ((uint32_t)kq << 24);
                }
                if (lane == 31) s_item[1] = (uint32_t)bincl;
            }
            __syncthreads();
            for (int rd = 0; rd < nrounds; rd++) {             // every thread moves the entries of the rounds' orders
                const uint16_t *sg = s_seg + rd * (BA_IN_NBKT + 1);
                const uint16_t *od = s_ordr + (size_t)rd * BA_NT;
                for (int idx = tid; idx < (int)sg[BA_IN_NBKT]; idx += BA_NT) {
                    int kq = 0;                                // the bucket of position idx: largest kq with sg[kq] <= idx
#pragma unroll
                    for (int st = BA_IN_NBKT / 2; st > 0; st >>= 1)
                        if ((int)sg[kq + st] <= idx) kq += st;
                    const int node = rd * BA_NT + od[idx], at = s_gstart[kq] + s_roff[rd * BA_IN_NBKT + kq] + (idx - (int)sg[kq]);
                    s_order[at] = (uint16_t)node;
                    if (MODE == IN_SWEEP) {
                        const uint32_t kk = s_rec[node].info >> 16;
                        s_skey[at] = (uint16_t)((s_rec[node].id & 0xffu) | ((kk < 15u ? kk : 15u) << 8));
                    }
                }
            }
            if (eps_fact) ba_cp_async_wait_all();              // this thread's c(y')
            __syncthreads();

            // ================= G sums of the pairs (v, empty) =================
            // A node y' of length k adds c(y') alpha_s to G(sigma_s) for s = 0 .. min(k, m).  Every sum has one owner
            // thread, which walks the two buckets of its class in their (stable) order: no atomics, one fixed order.
            // |w| >= 5: the thread of code(w) takes the nodes of class w mod 16 that end in w.  |w| <= 4: G(w) is the sum
            // over the classes that end in w of P(class, s) = sum over the class's nodes of length >= s; the 80 P's have
            // owners of their own (threads 480..511, then 0..47) and are added up in the epilogue.
            if (eps_fact) {
                auto scan = [&](int s, int cl, uint32_t wval, int dst) {
                    const uint32_t mask = (1u << s) - 1u;
                    double g = 0.0;
                    for (int part = 0; part < 2; part++) {
                        const int i0 = s_gstart[part * BA_NCLS + cl], i1 = s_gstart[part * BA_NCLS + cl + 1];
                        for (int i = i0; i < i1; i++) {
                            const uint32_t key = s_skey[i];    // one independent load per node; the record only on a match
                            if ((int)(key >> 8) >= s && (key & mask) == wval) {
                                const int node = s_order[i];
                                g = fma((double)s_rec[node].a[s], s_c[node], g);
                            }
                        }
                    }
                    s_G[dst] += g;
                };
                if (tid < 480) {
                    const uint32_t code = 32u + (uint32_t)tid;
                    const int s = ba_len_of_code(code);
                    const uint32_t wval = code - (1u << s);
                    scan(s, (int)(wval & (BA_NCLS - 1)), wval, (int)code);
                }
                if (tid >= 480 || tid < 5 * BA_NCLS - 32) {
                    const int j = (tid >= 480) ? tid - 480 : 32 + tid, cl = j / 5, s = j % 5;
                    scan(s, cl, (uint32_t)cl & ((1u << s) - 1u), 512 + j);
                }
            }

            // ================= phase B: batches of one class =================
            const int nbatch = (int)s_item[1];
            int st_cls = -1, st_sb = 0, cp_cls = -1, cp_sb = 0;     // slice double buffer: staging side, computing side
            // Staging is the work of warp 0 alone; the other warps meet it only through the FULL / EMPTY barriers of the
            // two buffers, so a warp runs up to one batch ahead of the slowest one and nobody waits at a CTA barrier.
            auto stage = [&](int j) {                          // half rows, slices and alphas of batch j (warp 0, lane i = node i)
                const uint32_t bi = s_batch[j], g = gb + (uint32_t)j;
                const int start = (int)(bi & 0xffffu), len = (int)((bi >> 16) & 0xffu), buf = (int)(g & 1u);
                const int scls = (int)(bi >> 24) & (BA_NCLS - 1);
                // every warp has left the batch that used this buffer, its slice buffer and its rider sums before
                if (g >= 2u) ba_mbar_wait(sEmpty + 8u * buf, ((g >> 1) - 1u) & 1u);
                const bool newcls = scls != st_cls;            // a new class: its slices of B_4..B_7 (by the sigma bits 4..6)
                if (newcls) { st_cls = scls; st_sb ^= 1; }     // of the riders and, for b = 0, of the pairs (v, empty)
                const uint32_t rs_bytes = (MODE == IN_SWEEP) ? 0u : 32u * (uint32_t)a.g.nr, es_bytes = (eps_enum && m == BA_MLOW) ? (8u << BA_MLOW) * 4u : 0u;
                const bool row = MODE == IN_SWEEP && lane < len && (bi >> 24) < BA_NCLS;
                uint32_t tx = row ? (uint32_t)nv * 8u : 0u;
                if (newcls && lane == 0) tx += rs_bytes + es_bytes;
                if (newcls && eps_enum && m != BA_MLOW) {      // n < 8: the rows of the slice are shorter than their pitch
                    const uint32_t *src = a.EPSH + (size_t)scls * 8 * nv;
                    for (int e = lane; e < 8 * nv; e += 32)
                        s_slice[(size_t)st_sb * (8u << BA_MLOW) + (size_t)((e >> m) << BA_MLOW) + (size_t)(e & (nv - 1))] = __ldg(src + e);
                }
                const NodeRec *rcp = nullptr;
                if (lane < len) {
                    const int node = s_order[start + lane];
                    rcp = &s_rec[node];
                    s_bal[buf * BA_RB_IN + lane] = ba_make_bal(*rcp, (uint32_t)node);
                }
                // the lane's arrival carries the bytes of its bulk copies
                if (tx) ba_mbar_arrive_expect_tx(sFull + 8u * buf, tx); else ba_mbar_arrive(sFull + 8u * buf);
                if (newcls && lane == 0) {
                    if (rs_bytes) ba_bulk_g2s(ba_smem_addr(s_rslice) + (uint32_t)st_sb * rs_bytes, a.g.R8 + ((size_t)scls * 2 + b) * 8 * a.g.nr, rs_bytes, sFull + 8u * buf);
                    if (es_bytes) ba_bulk_g2s(ba_smem_addr(s_slice) + (uint32_t)st_sb * es_bytes, a.EPSH + (size_t)scls * 8 * nv, es_bytes, sFull + 8u * buf);
                }
                if (row)                                       // the half row c(y'.b.t), all t, is row (code(y'), b) of crow: one bulk copy
                    ba_bulk_g2s(sRows + (uint32_t)(buf * BA_RB_IN + lane) * BA_ROWB, a.crow + (((((size_t)rcp->id) << 1) | (size_t)b) << m),
                                (uint32_t)nv * 8u, sFull + 8u * buf);
            };
            auto flush = [&](int j) {                          // thread v collects the rider sums of batch j
                if (MODE == IN_SWEEP) {                        // the owner of w collects the deep-part sums of its splits
                    if (tid >= 480) return;
                    const uint2 gm = s_g2map[b * 480 + tid];
                    if ((gm.x | gm.y) == 0u) return;
                    const uint32_t want = 0x80u | (s_batch[j] >> 24);
                    const double *rs = s_rsum + (size_t)((gb + (uint32_t)j) & 3u) * 2 * BA_G2_NT;
#pragma unroll
                    for (int q = 0; q < 4; q++) {
                        const uint32_t e = (((q >> 1) ? gm.y : gm.x) >> (16 * (q & 1))) & 0xffffu;
                        if ((e >> 8) == want) acc_g2 += rs[e & 0xffu] + rs[BA_G2_NT + (e & 0xffu)];
                    }
                    return;
                }
                if (MODE != IN_HC) return;
                if (tid >= nv) return;
                if ((s_batch[j] >> 24) >= BA_NCLS) return;     // a batch without list b has no riders
                const int cls = (int)(s_batch[j] >> 24), rbuf = (int)((gb + (uint32_t)j) & 3u);
                const uint16_t *cs = a.g.r_csr + (size_t)(cls * 2 + b) * (nv + 1) + tid;
                const int e0 = cs[0], e1 = cs[1];
                for (int e = e0; e < e1; e++) acc_rid += s_rsum[((size_t)rbuf * 2) * a.g.nr + e] + s_rsum[((size_t)rbuf * 2 + 1) * a.g.nr + e];
            };
            if (warp == 0 && nbatch > 0) stage(0);
            for (int j = 0; j < nbatch; j++) {
                const uint32_t bi = s_batch[j];
                const int len = (int)((bi >> 16) & 0xffu), cls = (int)(bi >> 24) & (BA_NCLS - 1), kind = (int)(bi >> 28), buf = (int)((gb + (uint32_t)j) & 1u);
                if (cls != cp_cls) { cp_cls = cls; cp_sb ^= 1; }
                uint32_t eB0 = 0u;                             // 1 | B_1..B_3 of the pair (ev, empty): a constant of the class
                if (eps_enum) eB0 = __ldg(a.EPS8 + (size_t)cls * nv + ev).x;
                // the slots' B_s do not depend on the staged rows: fetch them before waiting
                uint32_t Bp[BA_NSLOT];
#pragma unroll
                for (int k = 0; k < BA_KG; k++) {
                    uint4 bb = make_uint4(0u, 0u, 0u, 0u);
                    if (kind == 0) bb = __ldg(a.g.GB + (((size_t)cls * 2 + b) * BA_KG + k) * BA_NT + tid);
                    Bp[k * BA_GP] = bb.x; Bp[k * BA_GP + 1] = bb.y; Bp[k * BA_GP + 2] = bb.z; Bp[k * BA_GP + 3] = bb.w;
                }
                ba_mbar_wait(sFull + 8u * buf, ((gb + (uint32_t)j) >> 1) & 1u);     // rows, slices and records of batch j have landed
                if (warp == 0 && j + 1 < nbatch) stage(j + 1);
                // the rider sums of batch j-2: batch j was staged after every warp had left j-2, and no warp enters
                // j+2 (which takes their place) before this warp has left j
                if (j > 1) flush(j - 2);
                const uint32_t rowbase = sRows + (uint32_t)(buf * BA_RB_IN) * BA_ROWB;
                const BalRec *bal = s_bal + buf * BA_RB_IN;
                bool big = false;
                if (may_big) big = __any_sync(0xffffffffu, lane < len && bal[lane].big != 0u);
                // ---- the pair (v, empty) of every node of the batch: thread (v, node) -----------------------------
                if (eps_enum && (kind == 1 || klen < 0)) {
                    const uint32_t sv8 = (m == 8) ? (uint32_t)ev : 0xffffffffu;      // B_8 = [sigma_8 = v] (m = 8 only)
                    const uint32_t *sl = s_slice + (size_t)cp_sb * (8u << BA_MLOW) + ev;     // [sigma bits 4..6][v]
                    {
                        for (int i = esub; i < len; i += epn) {
                            const NodeRec &rc = s_rec[bal[i].node];
                            const uint32_t cy = rc.id;
                            const int k = (int)(rc.info >> 16);
                            const uint32_t emb = big ? ba_chain9_wide(rc.a, eB0, sl[((cy >> 4) & 7u) << BA_MLOW], (cy & 255u) == sv8)
                                                     : ba_chain9(bal[i].a01, bal[i].a23, bal[i].a45, bal[i].a67, bal[i].a8, eB0, sl[((cy >> 4) & 7u) << BA_MLOW], (cy & 255u) == sv8);
                            if (MODE == IN_HC) {
                                const double wk = s_w[k];
                                if (wk != 0.0) acc_eps = fma(wk, ba_elog2e(emb, a.elog, s_elog) - (double)emb * s_lebar[k], acc_eps);
                            } else if (MODE == IN_DEBUG) {
                                if (((u << m) | (uint32_t)ev) == a.dbg_x) a.dbg_out[cy - 1u] = emb;
                            } else {
                                cnt_terms += 1ull; cnt_emb += emb;
                            }
                        }
                    }
                }
                if (kind == 0) {
                if ((cls & 1) != cur_sc) {                     // the other schedule: swap the accumulators, reload the slot map
                    if (MODE == IN_SWEEP || MODE == IN_HC) {
                        if (cur_sc >= 0) {
#pragma unroll
                            for (int s = 0; s < BA_NSLOT; s++) park[((size_t)cur_sc * BA_NSLOT + s) * BA_NT] = acc[s];
                            parked |= 1u << cur_sc;
                        }
#pragma unroll
                        for (int s = 0; s < BA_NSLOT; s++) acc[s] = ((parked >> (cls & 1)) & 1u) ? park[((size_t)(cls & 1) * BA_NSLOT + s) * BA_NT] : 0.0;
                    }
                    cur_sc = cls & 1;
                    wmeta = a.g.GW[((size_t)cur_sc * 2 + b) * (BA_NT / 32) + warp];
#pragma unroll
                    for (int k = 0; k < BA_KG; k++) gaddr[k] = __ldg(a.g.GA + (((size_t)cur_sc * 2 + b) * BA_KG + k) * BA_NT + tid);
                }
                // ---- the thread's pair slots ---------------------------------------------------------------
                if (MODE == IN_HC && !big) {
                    // the slots of the thread against the nodes of the batch, as in the sweep, with the term
                    // w_k (emb log2 emb - emb log2 ebar_k) instead of emb * operand (|z| is a constant of the group)
                    int jz[BA_KG];
#pragma unroll
                    for (int g = 0; g < BA_KG; g++) jz[g] = ba_len_of_code(ba_z_of_tail((uint32_t)b, gaddr[g] >> 3));
#pragma unroll 2
                    for (int i = 0; i < len; i++) {
                        const uint2 al = *(const uint2 *)&bal[i];
                        const int k = ba_len_of_code(bal[i].id);
#pragma unroll
                        for (int g = 0; g < BA_KG; g++) {
                            const double wk = s_w[k + jz[g]], nlb = -s_lebar[k + jz[g]];
#pragma unroll
                            for (int q = 0; q < BA_GP; q++) {
                                uint32_t e = __dp2a_lo(al.x, Bp[g * BA_GP + q], 0u);
                                e = __dp2a_hi(al.y, Bp[g * BA_GP + q], e);
                                // exact u32 -> f64, spread over the conversion unit and the FP64 pipe as in the sweep
                                const double ed = (q == 0) ? ba_cvt<0>(e) : (q == 1) ? ba_cvt<1>(e) : (q == 2) ? ba_cvt<2>(e) : ba_cvt<3>(e);
                                const double gl = fma(ed, nlb, ba_elog2e(e, a.elog, s_elog));            // elog(0) = elog(1) = 0
                                acc[g * BA_GP + q] = fma(wk, gl, acc[g * BA_GP + q]);
                            }
                        }
                    }
                } else if (MODE == IN_SWEEP) {
                    uint32_t rb[BA_KG];
#pragma unroll
                    for (int k = 0; k < BA_KG; k++) rb[k] = rowbase + gaddr[k];
                    ba_group_batch(acc, Bp, rb, bal, s_rec, len, wmeta, big);
                } else {
                    for (int i = 0; i < len; i++) {
                        const NodeRec &rc = s_rec[bal[i].node];
                        const int k = (int)(rc.info >> 16);
#pragma unroll
                        for (int s = 0; s < BA_NSLOT; s++) {
                            const uint32_t bp = Bp[s];
                            if (!(bp & 0xffu)) continue;
                            const uint32_t emb = rc.a[0] * (bp & 0xffu) + rc.a[1] * ((bp >> 8) & 0xffu) + rc.a[2] * ((bp >> 16) & 0xffu) + rc.a[3] * (bp >> 24);
                            const uint32_t cz = ba_z_of_tail((uint32_t)b, gaddr[s / BA_GP] >> 3);
                            const int jz = ba_len_of_code(cz);
                            if (MODE == IN_HC) {
                                const double wk = s_w[k + jz];
                                if (wk != 0.0) acc[s] = fma(wk, ba_elog2e(emb, a.elog, s_elog) - (double)emb * s_lebar[k + jz], acc[s]);
                            } else if (MODE == IN_DEBUG) {
                                const uint32_t ov = a.g.GO[((((size_t)cur_sc * 2 + b) * BA_KG + s / BA_GP) * BA_GP + s % BA_GP) * BA_NT + tid];
                                if (((u << m) | ov) == a.dbg_x) a.dbg_out[((size_t)rc.id << jz) + (cz - (1u << jz)) - 1u] = emb;
                            } else {
                                cnt_terms += 1ull; cnt_emb += emb;
                            }
                        }
                    }
                }
                // ---- IN_SWEEP: the deep part of this batch, one target per thread (see acc_g2 above) --------
                if (MODE == IN_SWEEP && m >= 5) {
                    const int t2 = (BA_NT / 2 - 1) - (tid & (BA_NT / 2 - 1)), rh2 = tid / (BA_NT / 2);
                    if (t2 < BA_G2_NT) {
                        int s;
                        uint32_t ext, tc;                      // split, bits 4..s-1 of sigma_s, code(t) of z = b.t
                        if (t2 < 15) { s = 4; ext = 0u; tc = (uint32_t)t2 + 1u; }
                        else if (t2 < 29) { s = 5; ext = (uint32_t)(t2 - 15) / 7u; tc = (uint32_t)(t2 - 15) % 7u + 1u; }
                        else if (t2 < 41) { s = 6; ext = (uint32_t)(t2 - 29) / 3u; tc = (uint32_t)(t2 - 29) % 3u + 1u; }
                        else { s = 7; ext = (uint32_t)(t2 - 41); tc = 1u; }
                        const uint32_t pos = (tc == 1u) ? (uint32_t)b : tc, emask = (1u << (s - 4)) - 1u;
                        double g = 0.0;
                        if (s + 1 + ba_len_of_code(tc) <= m) {     // |sigma_s.z| <= m
                            const double *rrow = s_rows + (size_t)(buf * BA_RB_IN) * (BA_ROWB / 8) + pos;
                            for (int i = rh2; i < len; i += 2) {
                                const uint32_t cyi = bal[i].id;
                                if (ba_len_of_code(cyi) >= s && ((cyi >> 4) & emask) == ext) {
                                    uint32_t al;
                                    if (big) al = s_rec[bal[i].node].a[s];
                                    else {
                                        const uint32_t w2 = (s < 6) ? bal[i].a45 : bal[i].a67;
                                        al = (s & 1) ? (w2 >> 16) : (w2 & 0xffffu);
                                    }
                                    g = fma(ba_u2d(al), rrow[(size_t)i * (BA_ROWB / 8)], g);
                                }
                            }
                        }
                        s_rsum[((size_t)((gb + (uint32_t)j) & 3u) * 2 + rh2) * BA_G2_NT + t2] = g;
                    }
                }
                // ---- riders: deep pairs of this class, one per thread ------------------------------------
                const int nr = (MODE == IN_SWEEP) ? 0 : a.g.r_cnt[cls * 2 + b];
                // two replicas of the rider set (threads 255 - e and 511 - e), each takes every other node
                const int re = (BA_NT / 2 - 1) - (tid & (BA_NT / 2 - 1)), rh = tid / (BA_NT / 2);
                if ((BA_NT / 2) - 32 * ((warp & (BA_NT / 64 - 1)) + 1) < nr) {
                    double s = 0.0;
                    if (re < nr) {
                        const uint4 rd = __ldg(a.g.R + ((size_t)cls * 2 + b) * a.g.nr + re);
                        const uint32_t ov = rd.y >> 16;
                        const uint32_t cz = ba_z_of_tail((uint32_t)b, rd.z >> 3);
                        const int jz = ba_len_of_code(cz);
                        const uint32_t *r8 = s_rslice + (size_t)cp_sb * 8 * a.g.nr + re;           // B_4..B_7 by sigma bits 4..6: the class's slice
                        if (MODE == IN_SWEEP && !big) {
                            const double *rrow = s_rows + (size_t)(buf * BA_RB_IN) * (BA_ROWB / 8) + (rd.z >> 3);
                            double r0 = 0.0, r1 = 0.0;         // two chains; this replica's nodes rh, rh + 2, ...
#pragma unroll 4
                            for (int i = rh; i < len; i += 4) {
                                const uint4 al = *(const uint4 *)&bal[i];
                                const uint32_t x8 = r8[(size_t)((bal[i].id >> 4) & 7u) * a.g.nr];       // alpha_s = 0 beyond k
                                const uint32_t emb = ba_chain9(al.x, al.y, al.z, al.w, 0u, rd.x, x8, 0u);
                                r0 = fma(ba_u2d(emb), rrow[(size_t)i * (BA_ROWB / 8)], r0);
                                if (i + 2 < len) {
                                    const uint4 al2 = *(const uint4 *)&bal[i + 2];
                                    const uint32_t y8 = r8[(size_t)((bal[i + 2].id >> 4) & 7u) * a.g.nr];
                                    const uint32_t emb2 = ba_chain9(al2.x, al2.y, al2.z, al2.w, 0u, rd.x, y8, 0u);
                                    r1 = fma(ba_u2d(emb2), rrow[(size_t)(i + 2) * (BA_ROWB / 8)], r1);
                                }
                            }
                            s = r0 + r1;
                        } else {
                            for (int i = rh; i < len; i += 2) {
                                const BalRec bl = bal[i];
                                const uint32_t cy = bl.id;
                                const uint32_t x8 = r8[(size_t)((cy >> 4) & 7u) * a.g.nr];
                                const uint32_t emb = big ? ba_chain9_wide(s_rec[bl.node].a, rd.x, x8, 0u) : ba_chain9(bl.a01, bl.a23, bl.a45, bl.a67, 0u, rd.x, x8, 0u);
                                if (MODE == IN_SWEEP) {
                                    s = fma(ba_u2d(emb), ba_lds_f64(rowbase + (uint32_t)i * BA_ROWB + rd.z), s);
                                } else if (MODE == IN_HC) {
                                    const int k = (int)(s_rec[bl.node].info >> 16);
                                    const double wk = s_w[k + jz];
                                    if (wk != 0.0) s = fma(wk, ba_elog2e(emb, a.elog, s_elog) - (double)emb * s_lebar[k + jz], s);
                                } else if (MODE == IN_DEBUG) {
                                    if (((u << m) | ov) == a.dbg_x) a.dbg_out[((size_t)cy << jz) + (cz - (1u << jz)) - 1u] = emb;
                                } else {
                                    cnt_terms += 1ull; cnt_emb += emb;
                                }
                            }
                        }
                    }
                    if ((MODE == IN_SWEEP || MODE == IN_HC) && re < nr) s_rsum[((size_t)((gb + (uint32_t)j) & 3u) * 2 + rh) * a.g.nr + re] = s;
                }
                }                                              // kind == 0
                __syncwarp();
                if (lane == 0) ba_mbar_arrive(sEmpty + 8u * buf);      // this warp has left batch j
            }
            if (nbatch > 0) {
                __syncthreads();                               // rider sums of the last two batches are visible
                if (nbatch > 1) flush(nbatch - 2);
                flush(nbatch - 1);
            }
            gb += (uint32_t)nbatch;
        }

        // ---- epilogue: thread v owns x = u.v ------------------------------------------------------------
        __syncthreads();                                       // all rows consumed: the staging area becomes s_acc
        if (MODE == IN_SWEEP || MODE == IN_HC) {
            // the accumulators of both schedules to shared memory: the running one from registers, the other from its
            // parking place (zeros if it never ran)
#pragma unroll
            for (int sc = 0; sc < 2; sc++)
#pragma unroll
                for (int s = 0; s < BA_NSLOT; s++)
                    s_acc[((size_t)sc * BA_NSLOT + s) * BA_NT + tid] = (sc == cur_sc) ? acc[s] : ((parked >> sc) & 1u) ? park[((size_t)sc * BA_NSLOT + s) * BA_NT] : 0.0;
            double *s_aeps = s_rsum;                           // the rider sums are all flushed: their area takes acc_eps
            s_aeps[tid] = acc_eps;
            if (MODE == IN_SWEEP && tid < 480) s_G[32 + tid] += acc_g2;    // the owner's deep-part sums join its G(w)
            if (eps_fact && tid >= 480 && tid < 511) {         // G(w), |w| <= 4, from the P's of the classes that end in w
                const uint32_t code = (uint32_t)(tid - 479);
                const int s = ba_len_of_code(code);
                double g = 0.0;
                for (int cl = (int)(code - (1u << s)); cl < BA_NCLS; cl += 1 << s) g += s_G[512 + cl * 5 + s];
                s_G[code] = g;
            }
            __syncthreads();
            if (tid < nv) {
                double S = acc_rid;
                if (eps_enum)
                    for (int t = ev; t < BA_NT; t += nv) S += s_aeps[t];
                if (MODE == IN_SWEEP) {                        // sum_w G(w) emb(w, v) over the subsequences w of v
                    double se = 0.0;
                    for (uint32_t e = __ldg(a.LTV_off + tid), e1 = __ldg(a.LTV_off + tid + 1); e < e1; e++) {
                        const uint32_t ent = __ldg(a.LTV + e);
                        se = fma((double)(ent & 255u), s_G[ent >> 8], se);
                    }
                    S += se;
                }
                for (int sc = 0; sc < 2; sc++) {
                    const uint16_t *co = a.g.csr_off + ((size_t)sc * 2 + b) * (a.g.nown + 1) + tid, *ci = a.g.csr_idx + ((size_t)sc * 2 + b) * BA_NSLOT * BA_NT;
                    for (int q = co[0]; q < co[1]; q++) S += s_acc[(size_t)sc * BA_NSLOT * BA_NT + ci[q]];
                }
                a.S[(size_t)b * NX + (((size_t)u << m) | (size_t)tid)] = S;
            }
        }
        if (MODE == IN_DEBUG) break;
        __syncthreads();
        if (MODE == IN_HC) load_elog();                        // visible to all after the barriers of the next item's phase A
    }
    if (MODE == IN_COUNT) {
        atomicAdd(&a.cnt[0], cnt_terms);
        atomicAdd(&a.cnt[1], cnt_emb);
    }
}
