// ba_enum_out.cuh -- output sweep: q(y) = w_k sum_{x contains y} emb(y,x) p(x) as a
// GATHER over the length-n supersequences of y: every output has a
// single owner, nothing is accumulated with atomics.
//
// Work item = (high output prefix y' of length t <= h with code cy, list b); one persistent CTA per SM takes items
// from an atomic counter (short y' = many supersequences first).  Item (y', b) owns the outputs y'.z with z[0] = b
// (and, for b = 0, y' itself).  The class of an item is fixed, so the B_s of every pair are constants of the item.
// Per item, in super-batches of BA_NT nodes:
//   phase A  every thread UNRANKS one node: the r-th length-h supersequence u of y' (the paper's
//            subsetUnrank / RecSuperSeq, Alg. 5-6, with the G3 correction for the unmatched
//            tail; there are sum_{i<=h-t} C(h,i) of them by Lemma 6) and runs the textbook
//            integer DP  f[s] = emb(y'[0:t-s], u)  in registers; record {alpha_0..8, u, mask}.
//            For b = 0 the same thread adds the node's pair (v, empty) in factored form: sum_s alpha_s M(u, sigma_s),
//            M from k_low_tile (P:181 at the tile boundary).
//   sort     the nodes that carry list b are compacted (stable); the others are done (OUT_DEBUG / OUT_COUNT, which need
//            every emb on its own, let them follow in batches of the pair (v, empty) only).
//   phase B  batches of <= BA_RB_OUT nodes.  For node u the 2^m inputs p(u.*) -- the run of inputs whose low m
//            bits are free (SURVEY 7.2 "coalescing the gather") -- are one contiguous 2^m-double row, staged with
//            one bulk copy per row by warp 0 into a 3-stage ring whose FULL / EMPTY mbarriers are the only per-batch
//            synchronisation.  Every thread owns BA_KG groups of BA_GP pairs (ba_internal.h "GROUPS"): a group is one
//            v with up to 4 different z, so p(u.v) is read once per node and group, and
//                 1-2 IDP.2A (emb) + 1 exact u32->f64 + 1 DFMA            per (x,y) term.
//            The deep pairs (riders) use all nine B_s, read once per item from direct tables.
//   epilogue the slots of each z are added in a fixed order and written once:
//            Apart[y'][z] = sum_{u, v} emb(y'.z, u.v) p(u.v) over the nodes where y' is the longest
//            prefix of y'.z embeddable in u.
// k_out_final then adds, in a fixed order, the <= m+1 partials of each y:
//     A(y) = sum_j Apart[y[0:k-j]][y[k-j:]],   q(y) = w_k A(y),   c(y) = w_k log2(A(y)/ebar_k).
#pragma once
#include "ba_internal.h"

enum { OUT_SWEEP = 0, OUT_DEBUG = 1, OUT_COUNT = 2 };

#define BA_OUT_MAXB (4 + BA_NT / BA_RB_OUT)
#define BA_OUT_NSTG 3                                       // stages of the operand-row ring

__constant__ uint32_t c_binom[BA_NMAX_I + 1][BA_NMAX_I + 1];

struct OutArgs {
    KConst kc;
    GroupDev g;                // schedule of the output sweep (owner = code(z), operand position = v)
    const uint2 *EPS8;         // [256][2^m]: B(sigma_s, v), s = 1..8, of the pair (v, empty)
    const double *p;           // NX
    const double *M;           // OUT_SWEEP: [2^{m+1}][2^h] M(u, w) = sum_v p(u.v) emb(w, v) at [code(w)][u] (k_low_tile)
    double *Apart;             // (2^{h+1}-1) * (2^{m+1}-1)
    unsigned int *counter;
    int sym;                   // 1: q(y) = q(~y): prefixes y' with leading symbol 1 are skipped (k_out_final mirrors them)
    uint32_t dbg_item;         // OUT_DEBUG: code of y'
    uint32_t dbg_cz;           // OUT_DEBUG: code of z
    uint32_t *dbg_out;         // OUT_DEBUG: NX zero-filled
    unsigned long long *cnt;   // OUT_COUNT
};

struct OutSmem { size_t rec, rows, bal, mbar, order, wcnt, bstart, batch, red, binom, item, total; };

__host__ __device__ static inline OutSmem enum_out_smem(int nr) {
    OutSmem s;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 15) & ~(size_t)15; return at; };
    s.rec = take((size_t)BA_NT * sizeof(NodeRec));
    size_t rows = (size_t)BA_OUT_NSTG * BA_RB_OUT * BA_ROWB, ac = ((size_t)BA_NSLOT * BA_NT + (size_t)nr) * 8;
    s.rows = take(rows > ac ? rows : ac);                  // the epilogue's accumulator staging aliases the rows
    s.bal = take((size_t)BA_OUT_NSTG * BA_RB_OUT * sizeof(BalRec));
    s.mbar = take((size_t)2 * BA_OUT_NSTG * 8);            // FULL and EMPTY barrier of every stage
    s.order = take((size_t)BA_NT * 2);
    s.wcnt = take((size_t)(BA_NT / 32) * 2 * 2);
    s.bstart = take(3 * 2);
    s.batch = take((size_t)BA_OUT_MAXB * 4);
    s.red = take(32 * 8);
    s.binom = take((size_t)(BA_HMAX + 1) * (BA_HMAX + 2) * 4);   // C(a, w), a <= h: per-lane indices (constant memory would serialise)
    s.item = take(16);
    s.total = o;
    return s;
}

template <int MODE>
__global__ void __launch_bounds__(BA_NT, 1) k_enum_out(const __grid_constant__ OutArgs a) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int m = a.kc.m, h = a.kc.h, nv = 1 << m;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const OutSmem L = enum_out_smem(a.g.nr);
    const uint32_t NZ = (2u << m) - 1u;

    NodeRec *s_rec = (NodeRec *)(smem + L.rec);
    double *s_rows = (double *)(smem + L.rows);
    double *s_acc = s_rows;                                 // epilogue only
    BalRec *s_bal = (BalRec *)(smem + L.bal);
    uint16_t *s_order = (uint16_t *)(smem + L.order);
    uint16_t *s_wcnt = (uint16_t *)(smem + L.wcnt);
    uint16_t *s_bstart = (uint16_t *)(smem + L.bstart);
    uint32_t *s_batch = (uint32_t *)(smem + L.batch);
    double *s_red = (double *)(smem + L.red);
    uint32_t *s_item = (uint32_t *)(smem + L.item);        // [0] item, [1] number of batches
    uint32_t (*s_binom)[BA_HMAX + 2] = (uint32_t (*)[BA_HMAX + 2])(smem + L.binom);
    for (int i = tid; i < (BA_HMAX + 1) * (BA_HMAX + 2); i += BA_NT)
        s_binom[i / (BA_HMAX + 2)][i % (BA_HMAX + 2)] = c_binom[i / (BA_HMAX + 2)][i % (BA_HMAX + 2)];

    const uint32_t sRows = ba_smem_addr(s_rows), sBal = ba_smem_addr(s_bal);
    const uint32_t sFull = ba_smem_addr(smem + L.mbar), sEmpty = sFull + BA_OUT_NSTG * 8u;
    if (tid == 0) {
        for (int i = 0; i < BA_OUT_NSTG; i++) {
            ba_mbar_init(sFull + 8u * i, 32u);              // the 32 lanes of the staging warp; the rows count in bytes (complete_tx)
            ba_mbar_init(sEmpty + 8u * i, BA_NT);           // per thread: finished reading the stage
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    uint32_t gb = 0;                                        // batches staged so far by this CTA (uniform)
    const int ev = tid & (nv - 1);                          // v of this thread's empty-z pairs
    const int esub = tid >> m, epn = BA_NT >> m;
    const bool may_big = h > 18;                            // C(h, h/2) >= 2^16 first at h = 19
    __syncthreads();

    unsigned long long cnt_terms = 0, cnt_emb = 0;
    const uint32_t n_items = (h >= 31) ? 0xffffffffu : ((2u << h) - 1u);   // codes 1 .. 2^{h+1}-1

    for (;;) {
        if (tid == 0) {
            uint32_t it;
            if (MODE == OUT_DEBUG) {
                const uint32_t cz = a.dbg_cz;
                it = ((a.dbg_item - 1u) << 1) | ((cz >= 2u) ? ((cz >> (ba_len_of_code(cz) - 1)) & 1u) : 0u);
            } else it = atomicAdd(a.counter, 1u);
            s_item[0] = it;
        }
        __syncthreads();
        const uint32_t it = s_item[0];
        const uint32_t cy = (it >> 1) + 1u;
        const int b = (int)(it & 1u);
        if (cy > n_items) break;
        if (MODE == OUT_DEBUG && blockIdx.x != 0) break;
        const int t = ba_len_of_code(cy);
        const uint32_t yv = cy - (1u << t);
        if (a.sym && t >= 1 && ((cy >> (t - 1)) & 1u)) { __syncthreads(); continue; }   // served by its complement
        // exact channel BDC_{n,klen}: this prefix reaches the outputs of length t .. t+m only; length t is the pair
        // (v, empty) alone, which item (y', 0) serves
        const int klen = (MODE == OUT_SWEEP) ? a.kc.klen : -1;
        if (klen >= 0 && (klen < t || klen > t + m || (klen == t && b == 1))) { __syncthreads(); continue; }
        const bool do_eps = (b == 0) && (klen < 0 || klen == t);
        const bool do_grp = (klen != t);
        const int cls = (int)(cy & (BA_NCLS - 1));
        const int Lc = t < 8 ? t : 8;
        uint32_t R = 0;                                        // number of supersequences (Lemma 6)
        for (int w = 0; w <= h - t; w++) R += c_binom[h][w];

        // ---- per item: the thread's pair slots, all nine B_s of the eps pair (v = ev) and of its rider ----------
        const size_t sb = (size_t)cls * 2 + b;      // the schedule of the item's class and list
        const int wmeta = a.g.GW[sb * (BA_NT / 32) + warp];
        uint32_t Bp[BA_NSLOT], gaddr[BA_KG];
#pragma unroll
        for (int k = 0; k < BA_KG; k++) {
            const uint4 bb = __ldg(a.g.GB + (((size_t)cls * 2 + b) * BA_KG + k) * BA_NT + tid);
            Bp[k * BA_GP] = bb.x; Bp[k * BA_GP + 1] = bb.y; Bp[k * BA_GP + 2] = bb.z; Bp[k * BA_GP + 3] = bb.w;
            gaddr[k] = __ldg(a.g.GA + (sb * BA_KG + k) * BA_NT + tid);
        }
        // The pair (v, empty) of a node.  OUT_SWEEP: sum_v p(u.v) emb(y', u.v) = sum_s alpha_s M(u, sigma_s) (P:181 at
        // the tile boundary; M from k_low_tile), formed in phase A by the thread that unranks the node: no row, no batch.
        // OUT_DEBUG / OUT_COUNT enumerate its 2^m terms one by one in phase B (eps_enum).
        const bool eps_enum = do_eps && MODE != OUT_SWEEP;
        const int Lm = t < m ? t : m;                          // sigma_s, s <= Lm: B(sigma_s, v) = 0 for s > m
        uint32_t eB0 = 0, eB1 = 0, eB2 = 0;                    // B(sigma_s, ev): B_0 = 1; alpha_s = 0 beyond t
        if (eps_enum) {
            const uint2 e8 = __ldg(a.EPS8 + (size_t)(cy & 255u) * nv + ev);
            eB0 = e8.x; eB1 = e8.y; eB2 = (m == 8 && (cy & 255u) == (uint32_t)ev) ? 1u : 0u;   // B_8 = [sigma_8 = v]
        }
        const int nr = a.g.r_cnt[cls * 2 + b];
        const int re = BA_NT - 1 - tid;                        // riders sit on the last warps
        uint32_t rB0 = 0, rB1 = 0, rB2 = 0, roff = 0, rown = 0;
        if (re < nr) {
            const uint4 rd = __ldg(a.g.R + ((size_t)cls * 2 + b) * a.g.nr + re);
            const uint32_t x8 = __ldg(a.g.R8 + (((size_t)cls * 2 + b) * 8 + ((cy >> 4) & 7u)) * a.g.nr + re);
            rB0 = rd.x; rB1 = x8; rB2 = 0u;                     // B_0..3, B_4..7; B_8 = 0 (|z| >= 1)
            roff = rd.z; rown = rd.y >> 16;
        }

        double acc[BA_NSLOT];
#pragma unroll
        for (int s = 0; s < BA_NSLOT; s++) acc[s] = 0.0;
        double acc_eps = 0.0, acc_rid = 0.0;

        for (uint32_t base = 0; base < R; base += BA_NT) {
            __syncthreads();
            // ================= phase A: unrank supersequence base+tid of y', DP =================
            int key = -1;
            if (base + tid < R) {
                uint32_t w = 0, rem = base + tid;
                while (rem >= s_binom[h][w]) { rem -= s_binom[h][w]; w++; }
                // subsetUnrank(h, w, rem): S = the w positions that the leftmost embedding skips (Alg. 5)
                uint32_t S = 0;
                {
                    uint32_t ww = w, jj = rem;
                    for (int pp = 0; pp < h && ww > 0; pp++) {
                        const uint32_t cc = s_binom[h - pp - 1][ww - 1];
                        const bool in = jj < cc;
                        S |= (in ? 1u : 0u) << pp; ww -= in ? 1u : 0u; jj -= in ? 0u : cc;
                    }
                }
                // RecSuperSeq (Alg. 6 with the G3 reading): build u left to right
                uint32_t u = 0;
                int r = 0, ell = 0;
                // (branch-free: the lanes of a warp hold different S, so every branch on S would run both ways)
                for (int pp = 0; pp < h; pp++) {
                    const uint32_t skip = (S >> pp) & 1u;
                    const int rr = (r < t) ? r : t - 1;            // the symbol of y' in play: the next unmatched one, else the last
                    const uint32_t yb = (t == 0) ? 0u : ((yv >> (t - 1 - rr)) & 1u);
                    const uint32_t take = (skip ^ 1u) & (uint32_t)(r < t);
                    u = (u << 1) | (yb ^ skip);                    // a skipped position avoids that symbol, any other carries it
                    r += (int)take;
                    ell = (take && r == t) ? pp + 1 : ell;
                }
                // M(u, sigma_s) of the pair (v, empty): loaded now, used after the DP, which covers their latency
                double mv[BA_MLOW + 1];
#pragma unroll
                for (int s = 0; s <= BA_MLOW; s++) mv[s] = 0.0;
                if (MODE == OUT_SWEEP && do_eps) {
                    // M is laid out by w, then u: the threads of a warp unrank consecutive supersequences, which differ in
                    // their late positions, so one load touches a few sectors instead of 32
                    const double *Mu = a.M + u;
#pragma unroll
                    for (int s = 0; s <= BA_MLOW; s++)         // code(sigma_s) = 1 << s | last s symbols of y'
                        if (s <= Lm) mv[s] = __ldg(Mu + ((size_t)((1u << s) | (cy & ((1u << s) - 1u))) << h));
                }
                // f[s] = emb(y'[0:t-s], u): textbook DP over the positions of u, f indexed from the END of y'
                uint32_t f[BA_HMAX + 2];
#pragma unroll
                for (int s = 0; s <= BA_HMAX + 1; s++) f[s] = (s == t) ? 1u : 0u;
                const uint32_t tmask = (t >= 32) ? 0xffffffffu : ((1u << t) - 1u);
                for (int pp = 0; pp < h; pp++) {
                    const uint32_t ub = (u >> (h - 1 - pp)) & 1u;
                    const uint32_t mm = (ub ? yv : ~yv) & tmask;   // bit s: symbol t-s of y' equals u_pp
#pragma unroll
                    for (int s = 0; s < 8; s++)
                        if ((mm >> s) & 1u) f[s] += f[s + 1];
                    if (t > 8) {                               // mm has no bit at or above t: the tail of f stays as it is
#pragma unroll
                        for (int s = 8; s < 16; s++)
                            if ((mm >> s) & 1u) f[s] += f[s + 1];
                    }
                    if (t > 16) {
#pragma unroll
                        for (int s = 16; s <= BA_HMAX; s++)
                            if ((mm >> s) & 1u) f[s] += f[s + 1];
                    }
                }
                if (MODE == OUT_SWEEP && do_eps) {
                    double e = 0.0;
#pragma unroll
                    for (int s = BA_MLOW; s >= 0; s--) e = fma((double)f[s], mv[s], e);    // alpha_s = 0 beyond t
                    acc_eps += e;
                }
                NodeRec rc;
#pragma unroll
                for (int s = 0; s < 9; s++) rc.a[s] = f[s];
                const uint32_t miss0 = ba_nextpos(u, h, ell, 0u) >= h, miss1 = ba_nextpos(u, h, ell, 1u) >= h;
                rc.id = u;
                rc.info = miss0 | (miss1 << 1) | ((uint32_t)Lc << 8) | ((uint32_t)t << 16);
                s_rec[tid] = rc;
                const bool has = do_grp && (b ? miss1 : miss0);
                key = has ? 0 : (eps_enum ? 1 : -1);           // 0: pairs of list b (and eps); 1: the pair (v, empty) only
            }
            ba_bucket_sort<2>(key, s_order, s_wcnt, s_bstart);
            if (tid == 0) {                                    // batches: <= BA_RB_OUT consecutive nodes of one kind
                int nb = 0;
                for (int kq = 0; kq < 2; kq++)
                    for (int off = s_bstart[kq]; off < s_bstart[kq + 1]; off += BA_RB_OUT) {
                        const int len = (s_bstart[kq + 1] - off < BA_RB_OUT) ? (s_bstart[kq + 1] - off) : BA_RB_OUT;
                        s_batch[nb++] = (uint32_t)off | ((uint32_t)len << 16) | ((uint32_t)kq << 24);
                    }
                s_item[1] = (uint32_t)nb;
            }
            __syncthreads();

            // ================= phase B =================
            const int nbatch = (int)s_item[1];
            auto stage = [&](int j, uint32_t g) {              // p rows and alphas of batch j = ring batch g: warp 0 only
                if (warp != 0) return;
                const uint32_t bi = s_batch[j];
                const int start = (int)(bi & 0xffffu), len = (int)((bi >> 16) & 0xffu), buf = (int)(g % BA_OUT_NSTG);
                if (lane < len) {                              // lane i: node i of the batch
                    const int node = s_order[start + lane];
                    const NodeRec &rc = s_rec[node];
                    s_bal[buf * BA_RB_OUT + lane] = ba_make_bal(rc, (uint32_t)node);
                    if (MODE == OUT_SWEEP) {
                        // the whole row p(u.*) in one bulk copy (x fits 32 bits, n <= 30); its bytes complete the FULL
                        // barrier of the stage, the arrive releases the BalRec stored above
                        ba_mbar_arrive_expect_tx(sFull + 8u * buf, (uint32_t)nv * 8u);
                        ba_bulk_g2s(sRows + (uint32_t)(buf * BA_RB_OUT + lane) * BA_ROWB, a.p + ((size_t)rc.id << m), (uint32_t)nv * 8u, sFull + 8u * buf);
                    } else ba_mbar_arrive(sFull + 8u * buf);
                } else ba_mbar_arrive(sFull + 8u * buf);
            };
            for (int j = 0; j < BA_OUT_NSTG - 1 && j < nbatch; j++) stage(j, gb + j);
            for (int j = 0; j < nbatch; j++) {
                const uint32_t bi = s_batch[j];
                const uint32_t g = gb + (uint32_t)j;
                const int len = (int)((bi >> 16) & 0xffu), kind = (int)(bi >> 24), buf = (int)(g % BA_OUT_NSTG);
                ba_mbar_wait(sFull + 8u * buf, (g / BA_OUT_NSTG) & 1u);          // batch j staged by every thread
                const uint32_t rowbase = sRows + (uint32_t)(buf * BA_RB_OUT) * BA_ROWB;
                const BalRec *bal = s_bal + buf * BA_RB_OUT;
                const uint32_t balbase = sBal + (uint32_t)(buf * BA_RB_OUT) * (uint32_t)sizeof(BalRec);
                bool big = false;
                if (may_big) big = __any_sync(0xffffffffu, lane < len && bal[lane].big != 0u);

                // ---- the pair (v, empty) of every node: thread (v, node) ----------------------------------
                if (eps_enum) {
                    const double *erow = s_rows + (size_t)(buf * BA_RB_OUT) * (BA_ROWB / 8) + ev;
                    if (MODE == OUT_SWEEP && !big) {
                        double e0 = 0.0, e1 = 0.0;             // two chains; nodes esub, esub + epn, ...
#pragma unroll 4
                        for (int i = esub; i < len; i += 2 * epn) {
                            const uint4 al = *(const uint4 *)&bal[i];
                            const uint32_t emb = ba_chain9(al.x, al.y, al.z, al.w, bal[i].a8, eB0, eB1, eB2);
                            e0 = fma(ba_u2d(emb), erow[(size_t)i * (BA_ROWB / 8)], e0);
                            const int i2 = i + epn;
                            if (i2 < len) {
                                const uint4 al2 = *(const uint4 *)&bal[i2];
                                const uint32_t emb2 = ba_chain9(al2.x, al2.y, al2.z, al2.w, bal[i2].a8, eB0, eB1, eB2);
                                e1 = fma(ba_u2d(emb2), erow[(size_t)i2 * (BA_ROWB / 8)], e1);
                            }
                        }
                        acc_eps += e0 + e1;
                    } else {
                        for (int i = esub; i < len; i += epn) {
                            const uint32_t emb = big ? ba_chain9_wide(s_rec[bal[i].node].a, eB0, eB1, eB2)
                                                     : ba_chain9(bal[i].a01, bal[i].a23, bal[i].a45, bal[i].a67, bal[i].a8, eB0, eB1, eB2);
                            if (MODE == OUT_SWEEP) {
                                acc_eps = fma(ba_u2d(emb), erow[(size_t)i * (BA_ROWB / 8)], acc_eps);
                            } else if (MODE == OUT_DEBUG) {
                                if (a.dbg_cz == 1u) a.dbg_out[((size_t)bal[i].id << m) | (size_t)ev] = emb;
                            } else {
                                cnt_terms += 1ull; cnt_emb += emb;
                            }
                        }
                    }
                }
                if (kind == 0) {
                    // ---- the thread's pair slots ------------------------------------------------------------
                    if (MODE == OUT_SWEEP) {
                        uint32_t rb[BA_KG];
#pragma unroll
                        for (int k = 0; k < BA_KG; k++) rb[k] = rowbase + gaddr[k];
                        ba_group_batch(acc, Bp, rb, bal, s_rec, len, wmeta, big);
                    } else {
                        for (int i = 0; i < len; i++) {
                            const NodeRec &rc = s_rec[bal[i].node];
#pragma unroll
                            for (int s = 0; s < BA_NSLOT; s++) {
                                const uint32_t bp = Bp[s];
                                if (!(bp & 0xffu)) continue;
                                const uint32_t emb = rc.a[0] * (bp & 0xffu) + rc.a[1] * ((bp >> 8) & 0xffu) + rc.a[2] * ((bp >> 16) & 0xffu) + rc.a[3] * (bp >> 24);
                                if (MODE == OUT_DEBUG) {
                                    const uint32_t oz = a.g.GO[((sb * BA_KG + s / BA_GP) * BA_GP + s % BA_GP) * BA_NT + tid];
                                    if (oz == a.dbg_cz) a.dbg_out[((size_t)rc.id << m) | (size_t)(gaddr[s / BA_GP] >> 3)] = emb;
                                } else {
                                    cnt_terms += 1ull; cnt_emb += emb;
                                }
                            }
                        }
                    }
                    // ---- riders: deep pairs of this class, one per thread, all B_s static -----------------------
                    if (re < nr) {
                        const double *rrow = s_rows + (size_t)(buf * BA_RB_OUT) * (BA_ROWB / 8) + (roff >> 3);
                        if (MODE == OUT_SWEEP && !big) {
                            double r0 = 0.0, r1 = 0.0;
#pragma unroll 4
                            for (int i = 0; i < len; i += 2) {
                                const uint4 al = *(const uint4 *)&bal[i];
                                const uint32_t emb = ba_chain9(al.x, al.y, al.z, al.w, bal[i].a8, rB0, rB1, rB2);
                                r0 = fma(ba_u2d(emb), rrow[(size_t)i * (BA_ROWB / 8)], r0);
                                if (i + 1 < len) {
                                    const uint4 al2 = *(const uint4 *)&bal[i + 1];
                                    const uint32_t emb2 = ba_chain9(al2.x, al2.y, al2.z, al2.w, bal[i + 1].a8, rB0, rB1, rB2);
                                    r1 = fma(ba_u2d(emb2), rrow[(size_t)(i + 1) * (BA_ROWB / 8)], r1);
                                }
                            }
                            acc_rid += r0 + r1;
                        } else {
                            for (int i = 0; i < len; i++) {
                                const uint32_t emb = big ? ba_chain9_wide(s_rec[bal[i].node].a, rB0, rB1, rB2)
                                                         : ba_chain9(bal[i].a01, bal[i].a23, bal[i].a45, bal[i].a67, bal[i].a8, rB0, rB1, rB2);
                                if (MODE == OUT_SWEEP) {
                                    acc_rid = fma(ba_u2d(emb), rrow[(size_t)i * (BA_ROWB / 8)], acc_rid);
                                } else if (MODE == OUT_DEBUG) {
                                    if (rown == a.dbg_cz) a.dbg_out[((size_t)bal[i].id << m) | (size_t)(roff >> 3)] = emb;
                                } else {
                                    cnt_terms += 1ull; cnt_emb += emb;
                                }
                            }
                        }
                    }
                }
                ba_mbar_arrive(sEmpty + 8u * buf);             // this thread has finished reading the stage
                if (j + BA_OUT_NSTG - 1 < nbatch) {            // refill the stage of ring batch g-1 with batch j+NSTG-1
                    const uint32_t gn = g + BA_OUT_NSTG - 1;
                    if (warp == 0 && j >= 1) ba_mbar_wait(sEmpty + 8u * (gn % BA_OUT_NSTG), ((g - 1) / BA_OUT_NSTG) & 1u);
                    stage(j + BA_OUT_NSTG - 1, gn);
                }
            }
            gb += (uint32_t)nbatch;
        }

        // ---- epilogue: fixed-order reduction of the slots of each z, one write per (y', z) -----------------
        __syncthreads();                                       // rows are dead: the area becomes s_acc
        if (MODE == OUT_SWEEP) {
#pragma unroll
            for (int s = 0; s < BA_NSLOT; s++) s_acc[(size_t)s * BA_NT + tid] = acc[s];
            if (re < a.g.nr) s_acc[(size_t)BA_NSLOT * BA_NT + re] = acc_rid;
            double r0 = acc_eps;                               // z empty: block-wide sum, fixed tree
            for (int o = 16; o > 0; o >>= 1) r0 += __shfl_xor_sync(0xffffffffu, r0, o);
            if (lane == 0) s_red[warp] = r0;
            __syncthreads();
            double *dst = a.Apart + (size_t)(cy - 1u) * NZ;
            if (tid == 0 && b == 0) {
                double s = 0.0;
                for (int w = 0; w < BA_NT / 32; w++) s += s_red[w];
                dst[0] = s;
            }
            const uint16_t *co = a.g.csr_off + sb * (a.g.nown + 1), *ci = a.g.csr_idx + sb * BA_NSLOT * BA_NT;
            const uint16_t *cs = a.g.r_csr + ((size_t)cls * 2 + b) * (a.g.nown + 1);
            for (uint32_t cz = 2u + tid; cz <= NZ; cz += BA_NT) {      // cz = code(z), z not empty
                if ((int)((cz >> (ba_len_of_code(cz) - 1)) & 1u) != b) continue;
                double s = 0.0;
                for (int q = co[cz]; q < co[cz + 1]; q++) s += s_acc[ci[q]];
                for (int e = cs[cz]; e < cs[cz + 1]; e++) s += s_acc[(size_t)BA_NSLOT * BA_NT + e];
                dst[cz - 1u] = s;
            }
        }
        if (MODE == OUT_DEBUG) break;
        __syncthreads();
    }
    if (MODE == OUT_COUNT) {
        atomicAdd(&a.cnt[0], cnt_terms);
        atomicAdd(&a.cnt[1], cnt_emb);
    }
}
