// ba_enum_out.cuh -- output sweep: q(y) = w_k sum_{x contains y} emb(y,x) p(x) as a
// GATHER over the length-n supersequences of y: every output has a
// single owner, nothing is accumulated with atomics.
//
// Work item = a high output prefix y' (length t <= h, code cy); one persistent CTA per SM takes items
// from an atomic counter (short y' = many supersequences first).  The class of an item is fixed, so the
// B_s of every pair are constants of the whole item.  Per item, in super-batches of BA_NT nodes:
//   phase A  every thread UNRANKS one node: the r-th length-h supersequence u of y' (the paper's
//            subsetUnrank / RecSuperSeq, Alg. 5-6, with the G3 correction for the unmatched
//            tail; there are sum_{i<=h-t} C(h,i) of them by Lemma 6) and runs the textbook
//            integer DP  f[s] = emb(y'[0:t-s], u)  in registers; record {alpha_0..8, u, mask}.
//   sort     nodes are ranked, stably, by mask (which lists of non-empty z they carry).
//   phase B  batches of <= BA_RB_OUT nodes of one mask.  For node u the 2^m inputs p(u.*) -- the run
//            of inputs whose low m bits are free (SURVEY 7.2 "coalescing the gather") -- are one
//            contiguous 2^m-double row, staged with 16-byte cp.async into a 3-stage ring whose FULL / EMPTY
//            mbarriers are the only per-batch synchronisation (no CTA-wide barrier).  Pairs (v,z) are
//            dealt z-major: every thread owns BA_NC chunks of BA_C supersequences v of one z per list,
//            with one FP64 accumulator per chunk kept in a register for the whole item, and runs
//                 1-4 IMAD (emb) + 1 LDS.64 (p) + 1 exact u32->f64 + 1 DFMA             per (x,y) term.
//            The pair (v, empty) of every node and the deep pairs (riders) use all nine B_s, read once
//            per item from direct tables.
//   epilogue the chunks of each z are added in a fixed order and written once:
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
    const uint2 *EPS8;         // [256][2^m]: B(sigma_s, v), s = 1..8, of the pair (v, empty)
    const uint32_t *RO8;       // [cls][b][16][nro]: B_5..B_8 of a rider by the sigma bits 4..7
    const uint2 *FO;           // fast pairs [cls][b][c][q][tid]
    const uint4 *RO;           // riders [cls][b][nro]
    const uint16_t *ro_cnt;    // [cls][b]
    const uint16_t *ro_csr;    // [cls][b][2^{m+1} + 1] by code(z)
    int nro;
    const uint16_t *owner;     // [cls][b][c][tid] -> code(z)
    const uint16_t *csr_off;   // [cls][2^{m+1}] by code(z)-1
    const uint16_t *csr_idx;   // [cls][ncsr]
    int ncsr;
    const double *p;           // NX
    double *Apart;             // (2^{h+1}-1) * (2^{m+1}-1)
    unsigned int *counter;
    int sym;                   // 1: q(y) = q(~y): prefixes y' with leading symbol 1 are skipped (k_out_final mirrors them)
    uint32_t dbg_item;         // OUT_DEBUG: code of y'
    uint32_t dbg_cz;           // OUT_DEBUG: code of z
    uint32_t *dbg_out;         // OUT_DEBUG: NX zero-filled
    unsigned long long *cnt;   // OUT_COUNT
};

struct OutSmem { size_t rec, rows, bal, bnode, mbar, order, wcnt, bstart, batch, red, item, total; };

__host__ __device__ static inline OutSmem enum_out_smem(int m, int ncsr, int nro) {
    OutSmem s;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 15) & ~(size_t)15; return at; };
    s.rec = take((size_t)BA_NT * sizeof(NodeRec));
    size_t rows = (size_t)BA_OUT_NSTG * BA_RB_OUT * ((size_t)1 << m) * 8, ac = ((size_t)2 * BA_NC * BA_NT + 2 * (size_t)nro) * 8;
    s.rows = take(rows > ac ? rows : ac);                  // the epilogue's accumulator staging aliases the rows
    s.bal = take((size_t)BA_OUT_NSTG * BA_RB_OUT * 16);
    s.bnode = take((size_t)BA_OUT_NSTG * BA_RB_OUT * 2);
    s.mbar = take((size_t)2 * BA_OUT_NSTG * 8);            // FULL and EMPTY barrier of every stage
    s.order = take((size_t)BA_NT * 2);
    s.wcnt = take((size_t)(BA_NT / 32) * 4 * 2);
    s.bstart = take(5 * 2);
    s.batch = take((size_t)BA_OUT_MAXB * 4);
    (void)ncsr;
    s.red = take(32 * 8);
    s.item = take(16);
    s.total = o;
    return s;
}

template <int MODE>
__global__ void __launch_bounds__(BA_NT, 1) k_enum_out(const __grid_constant__ OutArgs a) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int m = a.kc.m, h = a.kc.h, nv = 1 << m;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const OutSmem L = enum_out_smem(m, a.ncsr, a.nro);
    const uint32_t ROWB = (uint32_t)nv * 8u;
    const uint32_t NZ = (2u << m) - 1u;

    NodeRec *s_rec = (NodeRec *)(smem + L.rec);
    double *s_rows = (double *)(smem + L.rows);
    double *s_acc = s_rows;                                 // epilogue only
    uint4 *s_bal = (uint4 *)(smem + L.bal);
    uint16_t *s_bnode = (uint16_t *)(smem + L.bnode);
    uint16_t *s_order = (uint16_t *)(smem + L.order);
    uint16_t *s_wcnt = (uint16_t *)(smem + L.wcnt);
    uint16_t *s_bstart = (uint16_t *)(smem + L.bstart);
    uint32_t *s_batch = (uint32_t *)(smem + L.batch);
    double *s_red = (double *)(smem + L.red);
    uint32_t *s_item = (uint32_t *)(smem + L.item);        // [0] item, [1] number of batches

    const uint32_t sRows = ba_smem_addr(s_rows);
    const uint32_t sFull = ba_smem_addr(smem + L.mbar), sEmpty = sFull + BA_OUT_NSTG * 8u;
    if (tid == 0) {
        for (int i = 0; i < BA_OUT_NSTG; i++) {
            ba_mbar_init(sFull + 8u * i, 2u * BA_NT);       // per thread: its copies landed + its plain stores done
            ba_mbar_init(sEmpty + 8u * i, BA_NT);           // per thread: finished reading the stage
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    uint32_t gb = 0;                                        // batches staged so far by this CTA (uniform)
    const int ev = tid & (nv - 1);                          // v of this thread's empty-z pairs
    const int esub = tid >> m, epn = BA_NT >> m;
    const int st_pc = tid & ((nv >> 1) - 1), st_i0 = tid >> (m - 1), st_step = BA_NT >> (m - 1);   // staging role
    const uint32_t st_src = 2u * (uint32_t)st_pc, st_dst = ba_swz(2u * (uint32_t)st_pc) * 8u;
    __syncthreads();

    unsigned long long cnt_terms = 0, cnt_emb = 0;
    const uint32_t n_items = (h >= 31) ? 0xffffffffu : ((2u << h) - 1u);   // codes 1 .. 2^{h+1}-1

    for (;;) {
        if (tid == 0) s_item[0] = (MODE == OUT_DEBUG) ? a.dbg_item : atomicAdd(a.counter, 1u) + 1u;
        __syncthreads();
        const uint32_t cy = s_item[0];
        if (cy > n_items) break;
        if (MODE == OUT_DEBUG && blockIdx.x != 0) break;
        const int t = ba_len_of_code(cy);
        const uint32_t yv = cy - (1u << t);
        if (a.sym && t >= 1 && ((cy >> (t - 1)) & 1u)) { __syncthreads(); continue; }   // served by its complement
        // exact channel BDC_{n,klen}: this prefix reaches the outputs of length t .. t+m only
        const int klen = (MODE == OUT_SWEEP) ? a.kc.klen : -1;
        if (klen >= 0 && (klen < t || klen > t + m)) { __syncthreads(); continue; }
        const int cls = (int)(cy & (BA_NCLS - 1));
        const int Lc = t < 8 ? t : 8;
        uint32_t R = 0;                                        // number of supersequences (Lemma 6)
        for (int w = 0; w <= h - t; w++) R += c_binom[h][w];

        // ---- per item: all nine B_s of the eps pair (v = ev) and of this thread's riders --------------------
        uint32_t Ee[9];                                        // B(sigma_s, ev); alpha_s = 0 beyond t
        {
            const uint2 e8 = __ldg(a.EPS8 + (size_t)(cy & 255u) * nv + ev);
            Ee[0] = 1u;
            Ee[1] = e8.x & 0xffu; Ee[2] = (e8.x >> 8) & 0xffu; Ee[3] = (e8.x >> 16) & 0xffu; Ee[4] = e8.x >> 24;
            Ee[5] = e8.y & 0xffu; Ee[6] = (e8.y >> 8) & 0xffu; Ee[7] = (e8.y >> 16) & 0xffu; Ee[8] = e8.y >> 24;
        }
        uint32_t rB[2][3], roff[2];                            // riders: B_0..B_8 packed 4+4+1 bytes, row offset
#pragma unroll
        for (int b = 0; b < 2; b++) {
            rB[b][0] = rB[b][1] = rB[b][2] = 0u; roff[b] = 0u;
            const int nr = a.ro_cnt[cls * 2 + b];
            if (BA_NT - 1 - tid < nr) {                        // riders sit on the last warps (two chunk slots only)
                const uint4 rd = __ldg(a.RO + ((size_t)cls * 2 + b) * a.nro + (BA_NT - 1 - tid));
                rB[b][0] = rd.x;
                roff[b] = rd.z;
                const uint32_t x8 = __ldg(a.RO8 + (((size_t)cls * 2 + b) * 16 + ((cy >> 4) & 15u)) * a.nro + (BA_NT - 1 - tid));
                const uint32_t hi = (rd.y & 0xffu) | (x8 << 8), b8 = x8 >> 24;     // B_4..B_7, B_8
                rB[b][1] = hi; rB[b][2] = b8;
            }
        }

        double acc[2][BA_NC];
#pragma unroll
        for (int b = 0; b < 2; b++)
#pragma unroll
            for (int c = 0; c < BA_NC; c++) acc[b][c] = 0.0;
        double acc_eps = 0.0, acc_rid[2] = {0.0, 0.0};

        for (uint32_t base = 0; base < R; base += BA_NT) {
            __syncthreads();
            // ================= phase A: unrank supersequence base+tid of y', DP =================
            int key = -1;
            if (base + tid < R) {
                uint32_t w = 0, rem = base + tid;
                while (rem >= c_binom[h][w]) { rem -= c_binom[h][w]; w++; }
                // subsetUnrank(h, w, rem): S = the w positions that the leftmost embedding skips (Alg. 5)
                uint32_t S = 0;
                {
                    uint32_t ww = w, jj = rem;
                    for (int pp = 0; pp < h && ww > 0; pp++) {
                        const uint32_t cc = c_binom[h - pp - 1][ww - 1];
                        if (jj < cc) { S |= 1u << pp; ww--; } else { jj -= cc; }
                    }
                }
                // RecSuperSeq (Alg. 6 with the G3 reading): build u left to right
                uint32_t u = 0;
                int r = 0, ell = 0;
                for (int pp = 0; pp < h; pp++) {
                    uint32_t bit;
                    if ((S >> pp) & 1u) {
                        if (t == 0) bit = 1u;
                        else { const int rr = (r < t) ? r : t - 1; bit = 1u ^ ((yv >> (t - 1 - rr)) & 1u); }
                    } else if (r < t) {
                        bit = (yv >> (t - 1 - r)) & 1u; r++;
                        if (r == t) ell = pp + 1;
                    } else {
                        bit = (t == 0) ? 0u : (yv & 1u);
                    }
                    u = (u << 1) | bit;
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
                    for (int s = 0; s <= BA_HMAX; s++)
                        if ((mm >> s) & 1u) f[s] += f[s + 1];
                }
                NodeRec rc;
#pragma unroll
                for (int s = 0; s < 9; s++) rc.a[s] = f[s];
                const uint32_t miss0 = ba_nextpos(u, h, ell, 0u) >= h, miss1 = ba_nextpos(u, h, ell, 1u) >= h;
                rc.id = u;
                rc.info = miss0 | (miss1 << 1) | ((uint32_t)Lc << 8) | ((uint32_t)t << 16);
                rc.pad = 0u;
                s_rec[tid] = rc;
                key = (int)(miss0 | (miss1 << 1));
            }
            ba_bucket_sort<4>(key, s_order, s_wcnt, s_bstart);
            if (tid == 0) {                                    // batches: <= BA_RB_OUT consecutive nodes of one mask
                int nb = 0;
                for (int kq = 0; kq < 4; kq++)
                    for (int off = s_bstart[kq]; off < s_bstart[kq + 1]; off += BA_RB_OUT) {
                        const int len = (s_bstart[kq + 1] - off < BA_RB_OUT) ? (s_bstart[kq + 1] - off) : BA_RB_OUT;
                        s_batch[nb++] = (uint32_t)off | ((uint32_t)len << 16) | ((uint32_t)kq << 24);
                    }
                s_item[1] = (uint32_t)nb;
            }
            __syncthreads();

            // ================= phase B =================
            const int nbatch = (int)s_item[1];
            auto stage = [&](int j, uint32_t g) {              // p rows, alpha_0..3 and node ids of batch j = ring batch g
                const uint32_t bi = s_batch[j];
                const int start = (int)(bi & 0xffffu), len = (int)((bi >> 16) & 0xffu), buf = (int)(g % BA_OUT_NSTG);
                if (MODE == OUT_SWEEP) {
                    // 16-byte pieces, 2^{m-1} per row: a thread always copies the same piece, of every st_step-th row
                    for (int i = st_i0; i < len; i += st_step) {
                        const uint32_t u = s_rec[s_order[start + i]].id;
                        ba_cp_async16(sRows + (uint32_t)(buf * BA_RB_OUT + i) * ROWB + st_dst, a.p + ((u << m) + st_src));   // x fits 32 bits (n <= 30)
                    }
                }
                if (tid < len) {
                    const int node = s_order[start + tid];
                    s_bal[buf * BA_RB_OUT + tid] = *(const uint4 *)&s_rec[node].a[0];
                    s_bnode[buf * BA_RB_OUT + tid] = (uint16_t)node;
                }
                ba_mbar_arrive_on_copies(sFull + 8u * buf);    // when this thread's rows have landed
                ba_mbar_arrive(sFull + 8u * buf);              // releases its plain stores above
            };
            for (int j = 0; j < BA_OUT_NSTG - 1 && j < nbatch; j++) stage(j, gb + j);
            for (int j = 0; j < nbatch; j++) {
                const uint32_t bi = s_batch[j];
                const uint32_t g = gb + (uint32_t)j;
                const int len = (int)((bi >> 16) & 0xffu), mask = (int)(bi >> 24), buf = (int)(g % BA_OUT_NSTG);
                // the pairs of a chunk do not depend on the staged rows: fetch the first slot before waiting, and
                // the next slot while the current one is computed (one exposed L2 latency per batch at most)
                const uint2 *F0 = a.FO + ((size_t)cls * 2 * BA_NC) * BA_C * BA_NT + tid;   // list 0; list 1 follows
                uint32_t nbp[BA_C], nad[BA_C];
                {
                    const uint2 *Ff = F0 + ((mask & 1) ? 0 : (size_t)BA_NC * BA_C * BA_NT);
#pragma unroll
                    for (int q = 0; q < BA_C; q++) { const uint2 pr = __ldg(Ff + (size_t)q * BA_NT); nbp[q] = pr.x; nad[q] = pr.y; }
                }
                ba_mbar_wait(sFull + 8u * buf, (g / BA_OUT_NSTG) & 1u);          // batch j staged by every thread
                const uint32_t rowbase = sRows + (uint32_t)(buf * BA_RB_OUT) * ROWB;
                const uint4 *bal = s_bal + buf * BA_RB_OUT;
                const uint16_t *bnode = s_bnode + buf * BA_RB_OUT;

                // ---- the pair (v, empty) of every node: thread (v, node) ----------------------------------
                for (int i = esub; i < len && (klen < 0 || klen == t); i += epn) {
                    const NodeRec &rc = s_rec[bnode[i]];
                    const uint4 r0 = *(const uint4 *)&rc.a[0], r1 = *(const uint4 *)&rc.a[4], r2 = *(const uint4 *)&rc.a[8];
                    const uint32_t emb = r0.x * Ee[0] + r0.y * Ee[1] + r0.z * Ee[2] + r0.w * Ee[3] + r1.x * Ee[4] +
                                         r1.y * Ee[5] + r1.z * Ee[6] + r1.w * Ee[7] + r2.x * Ee[8];
                    if (MODE == OUT_SWEEP) {
                        acc_eps = fma(ba_u2d(emb), ba_lds_f64(rowbase + (uint32_t)i * ROWB + ba_swz((uint32_t)ev) * 8u), acc_eps);
                    } else if (MODE == OUT_DEBUG) {
                        if (a.dbg_cz == 1u) a.dbg_out[((size_t)r2.y << m) | (size_t)ev] = emb;
                    } else {
                        cnt_terms += 1ull; cnt_emb += emb;
                    }
                }
#pragma unroll
                for (int b = 0; b < 2; b++) {
                    if (!((mask >> b) & 1) || klen == t) continue;
                    // ---- fast pairs -----------------------------------------------------------------------
#pragma unroll
                    for (int c = 0; c < BA_NC; c++) {
                        uint32_t bp[BA_C], ad[BA_C];
#pragma unroll
                        for (int q = 0; q < BA_C; q++) { bp[q] = nbp[q]; ad[q] = nad[q]; }
                        if (c + 1 < BA_NC || (b == 0 && (mask & 2))) {      // next slot: (b, c+1), else (1, 0)
                            const uint2 *Fn = F0 + (size_t)((c + 1 < BA_NC) ? (b * BA_NC + c + 1) : BA_NC) * BA_C * BA_NT;
#pragma unroll
                            for (int q = 0; q < BA_C; q++) { const uint2 pr = __ldg(Fn + (size_t)q * BA_NT); nbp[q] = pr.x; nad[q] = pr.y; }
                        }
                        if (MODE == OUT_SWEEP) {
                            acc[b][c] = ba_fast_chunk(acc[b][c], bal, rowbase, ROWB, len, bp, ad);
                        } else {
                            const uint32_t oz = a.owner[(((size_t)cls * 2 + b) * BA_NC + c) * BA_NT + tid];
                            for (int i = 0; i < len; i++) {
                                const uint4 al = bal[i];
                                const uint32_t u = s_rec[bnode[i]].id;
#pragma unroll
                                for (int q = 0; q < BA_C; q++) {
                                    if (!(bp[q] & 0xffu)) continue;
                                    const uint32_t emb = al.x * (bp[q] & 0xffu) + al.y * ((bp[q] >> 8) & 0xffu) + al.z * ((bp[q] >> 16) & 0xffu) + al.w * (bp[q] >> 24);
                                    if (MODE == OUT_DEBUG) {
                                        if (oz == a.dbg_cz) a.dbg_out[((size_t)u << m) | (size_t)ba_swz(ad[q] >> 3)] = emb;
                                    } else {
                                        cnt_terms += 1ull; cnt_emb += emb;
                                    }
                                }
                            }
                        }
                    }
                    // ---- riders: deep pairs of this class, one per thread, all B_s static -----------------------
                    const int nr = a.ro_cnt[cls * 2 + b];
                    if (BA_NT - 1 - tid < nr) {
                        const uint32_t x0 = rB[b][0], x1 = rB[b][1], b8 = rB[b][2];
                        const uint32_t oz = __ldg(a.RO + ((size_t)cls * 2 + b) * a.nro + (BA_NT - 1 - tid)).y >> 16;
                        double s = acc_rid[b];
                        for (int i = 0; i < len; i++) {
                            const NodeRec &rc = s_rec[bnode[i]];
                            const uint4 r0 = *(const uint4 *)&rc.a[0], r1 = *(const uint4 *)&rc.a[4], r2 = *(const uint4 *)&rc.a[8];
                            const uint32_t emb = r0.x * (x0 & 0xffu) + r0.y * ((x0 >> 8) & 0xffu) + r0.z * ((x0 >> 16) & 0xffu) +
                                                 r0.w * (x0 >> 24) + r1.x * (x1 & 0xffu) + r1.y * ((x1 >> 8) & 0xffu) +
                                                 r1.z * ((x1 >> 16) & 0xffu) + r1.w * (x1 >> 24) + r2.x * b8;
                            if (MODE == OUT_SWEEP) {
                                s = fma(ba_u2d(emb), ba_lds_f64(rowbase + (uint32_t)i * ROWB + roff[b]), s);
                            } else if (MODE == OUT_DEBUG) {
                                if (oz == a.dbg_cz) a.dbg_out[((size_t)r2.y << m) | (size_t)ba_swz(roff[b] >> 3)] = emb;
                            } else {
                                cnt_terms += 1ull; cnt_emb += emb;
                            }
                        }
                        acc_rid[b] = s;
                    }
                }
                ba_mbar_arrive(sEmpty + 8u * buf);             // this thread has finished reading the stage
                if (j + BA_OUT_NSTG - 1 < nbatch) {            // refill the stage of ring batch g-1 with batch j+NSTG-1
                    const uint32_t gn = g + BA_OUT_NSTG - 1;
                    if (j >= 1) ba_mbar_wait(sEmpty + 8u * (gn % BA_OUT_NSTG), ((g - 1) / BA_OUT_NSTG) & 1u);
                    stage(j + BA_OUT_NSTG - 1, gn);
                }
            }
            gb += (uint32_t)nbatch;
        }

        // ---- epilogue: fixed-order reduction of the chunks of each z, one write per (y', z) -----------------
        __syncthreads();                                       // rows are dead: the area becomes s_acc
        if (MODE == OUT_SWEEP) {
#pragma unroll
            for (int b = 0; b < 2; b++) {
#pragma unroll
                for (int c = 0; c < BA_NC; c++) s_acc[((size_t)b * BA_NC + c) * BA_NT + tid] = acc[b][c];
                if (BA_NT - 1 - tid < a.nro) s_acc[(size_t)2 * BA_NC * BA_NT + (size_t)b * a.nro + (BA_NT - 1 - tid)] = acc_rid[b];
            }
            double r0 = acc_eps;                               // z empty: block-wide sum, fixed tree
            for (int o = 16; o > 0; o >>= 1) r0 += __shfl_xor_sync(0xffffffffu, r0, o);
            if (lane == 0) s_red[warp] = r0;
            __syncthreads();
            double *dst = a.Apart + (size_t)(cy - 1u) * NZ;
            if (tid == 0) {
                double s = 0.0;
                for (int w = 0; w < BA_NT / 32; w++) s += s_red[w];
                dst[0] = s;
            }
            for (uint32_t zi = 1u + tid; zi < NZ; zi += BA_NT) {   // zi = code(z) - 1
                double s = 0.0;
                const uint16_t *co = a.csr_off + (size_t)cls * (2u << m) + zi, *ci = a.csr_idx + (size_t)cls * a.ncsr;
                for (int q = co[0]; q < co[1]; q++) s += s_acc[ci[q]];
                const uint32_t cz = zi + 1u;
                const int b = (int)((cz >> (ba_len_of_code(cz) - 1)) & 1u);
                const uint16_t *cs = a.ro_csr + ((size_t)cls * 2 + b) * ((2u << m) + 1u) + cz;
                for (int e = cs[0]; e < cs[1]; e++) s += s_acc[(size_t)2 * BA_NC * BA_NT + (size_t)b * a.nro + e];
                dst[zi] = s;
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
