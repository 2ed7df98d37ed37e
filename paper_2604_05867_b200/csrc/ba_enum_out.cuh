// ba_enum_out.cuh -- output sweep: q(y) = w_k sum_{x contains y} emb(y,x) p(x) as a
// GATHER over the length-n supersequences of y: every output has a
// single owner, nothing is accumulated with atomics.
//
// Work item = a high output prefix y' (length t <= h, code cy); one persistent CTA per SM takes items
// from an atomic counter (short y' = many supersequences first).  Per item:
//   phase A  every thread UNRANKS one node: the r-th length-h supersequence u of y' (the paper's
//            subsetUnrank / RecSuperSeq, Alg. 5-6, with the G3 correction for the unmatched
//            tail; there are sum_{i<=h-t} C(h,i) of them by Lemma 6) and runs the textbook
//            integer DP  f[s] = emb(y'[0:t-s], u)  in registers; record {alpha_0..8, u, mask}.
//   phase B  all threads walk the node list.  For node u the 2^m inputs p(u.*) -- the run of inputs
//            whose low m bits are free (SURVEY 7.2 "coalescing the gather") -- are one contiguous
//            2^m-double row, staged with 16-byte cp.async.  The pairs (v, z) of the node (ba_internal.h)
//            are dealt to the threads by a STATIC z-major schedule: chunks of BA_C supersequences v of
//            one z, so each thread keeps one FP64 accumulator per chunk in registers for the whole
//            item.  emb(y'.z, u.v) = sum_s alpha_s B(sigma_s.z, v).
//   epilogue the chunks of each z are added in a fixed order and written once:
//            Apart[y'][z] = sum_{u, v} emb(y'.z, u.v) p(u.v) over the nodes where y' is the longest
//            prefix of y'.z embeddable in u.
// k_out_final then adds, in a fixed order, the <= m+1 partials of each y:
//     A(y) = sum_j Apart[y[0:k-j]][y[k-j:]],   q(y) = w_k A(y),   c(y) = w_k log2(A(y)/ebar_k).
#pragma once
#include "ba_internal.h"

enum { OUT_SWEEP = 0, OUT_DEBUG = 1, OUT_COUNT = 2 };

__constant__ uint32_t c_binom[BA_NMAX_I + 1][BA_NMAX_I + 1];

struct OutArgs {
    KConst kc;
    const uint2 *Tz;           // z-major pairs
    const uint32_t *Wv;        // v-major W words
    const uint32_t *vbase;     // [2^m]
    const uint2 *desc;         // [2][BA_NC][BA_NT]
    const uint16_t *csr_off;   // [2^{m+1}] by code(z)-1
    const uint16_t *csr_idx;
    int nTz, nWv, ncsr;
    const double *p;           // NX
    double *Apart;             // (2^{h+1}-1) * (2^{m+1}-1)
    unsigned int *counter;
    uint32_t dbg_item;         // OUT_DEBUG: code of y'
    uint32_t dbg_cz;           // OUT_DEBUG: code of z
    uint32_t *dbg_out;         // OUT_DEBUG: NX zero-filled
    unsigned long long *cnt;   // OUT_COUNT
};

struct OutSmem { size_t Tz, Wv, rec, stage, csr_off, csr_idx, red, item, total; };

__host__ __device__ static inline OutSmem enum_out_smem(int m, int nTz, int nWv, int ncsr) {
    OutSmem s;
    size_t o = 0;
    s.Tz = o; o += ((size_t)nTz * 8 + 15) & ~(size_t)15;
    s.Wv = o; o += ((size_t)nWv * 4 + 15) & ~(size_t)15;
    s.rec = o;                                             // records + rows; the epilogue's accumulator staging aliases both
    size_t rr = (size_t)BA_NT * sizeof(NodeRec) + (size_t)BA_NSTAGE * ((size_t)1 << m) * 8;
    size_t ac = (size_t)2 * BA_NC * BA_NT * 8;
    o += rr > ac ? rr : ac;
    s.stage = s.rec + (size_t)BA_NT * sizeof(NodeRec);
    s.csr_off = o; o += (((size_t)2 << m) * 2 + 15) & ~(size_t)15;
    s.csr_idx = o; o += ((size_t)ncsr * 2 + 15) & ~(size_t)15;
    s.red = o; o += 32 * 8;
    s.item = o; o += 16;
    s.total = o;
    return s;
}

template <int MODE>
__global__ void __launch_bounds__(BA_NT, 1) k_enum_out(const __grid_constant__ OutArgs a) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int m = a.kc.m, h = a.kc.h, nv = 1 << m;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const OutSmem L = enum_out_smem(m, a.nTz, a.nWv, a.ncsr);
    const uint32_t ROWB = (uint32_t)nv * 8u;
    const uint32_t NZ = (2u << m) - 1u;

    uint2 *s_Tz = (uint2 *)(smem + L.Tz);
    uint32_t *s_Wv = (uint32_t *)(smem + L.Wv);
    NodeRec *s_rec = (NodeRec *)(smem + L.rec);
    double *s_acc = (double *)(smem + L.rec);               // epilogue only
    uint16_t *s_csr_off = (uint16_t *)(smem + L.csr_off);
    uint16_t *s_csr_idx = (uint16_t *)(smem + L.csr_idx);
    double *s_red = (double *)(smem + L.red);
    uint32_t *s_item = (uint32_t *)(smem + L.item);

    for (int i = tid; i < a.nTz; i += BA_NT) s_Tz[i] = a.Tz[i];
    for (int i = tid; i < a.nWv; i += BA_NT) s_Wv[i] = a.Wv[i];
    for (int i = tid; i < (2 << m); i += BA_NT) s_csr_off[i] = a.csr_off[i];
    for (int i = tid; i < a.ncsr; i += BA_NT) s_csr_idx[i] = a.csr_idx[i];

    uint2 dsc[2][BA_NC];
#pragma unroll
    for (int b = 0; b < 2; b++)
#pragma unroll
        for (int c = 0; c < BA_NC; c++) dsc[b][c] = a.desc[((size_t)b * BA_NC + c) * BA_NT + tid];
    const uint32_t sTz = ba_smem_addr(s_Tz);
    const uint32_t sWv = ba_smem_addr(s_Wv);
    const uint32_t sStage = ba_smem_addr(smem + L.stage);
    const int ev = tid & (nv - 1);
    const int esub = tid >> m;
    const int epn = (BA_NT >> m) < BA_GRP ? (BA_NT >> m) : BA_GRP;
    const uint32_t evb = sWv + a.vbase[ev] * 4u;
    __syncthreads();
    const uint32_t eW = s_Wv[a.vbase[ev] + 1];              // W of (v, empty)

    unsigned long long cnt_terms = 0, cnt_emb = 0;
    const uint32_t n_items = (h >= 31) ? 0xffffffffu : ((2u << h) - 1u);   // codes 1 .. 2^{h+1}-1

    for (;;) {
        if (tid == 0) *s_item = (MODE == OUT_DEBUG) ? a.dbg_item : atomicAdd(a.counter, 1u) + 1u;
        __syncthreads();
        const uint32_t cy = *s_item;
        if (cy > n_items) break;
        if (MODE == OUT_DEBUG && blockIdx.x != 0) break;
        const int t = ba_len_of_code(cy);
        const uint32_t yv = cy - (1u << t);
        uint32_t R = 0;                                        // number of supersequences (Lemma 6)
        for (int w = 0; w <= h - t; w++) R += c_binom[h][w];

        double acc[2][BA_NC];
#pragma unroll
        for (int b = 0; b < 2; b++)
#pragma unroll
            for (int c = 0; c < BA_NC; c++) acc[b][c] = 0.0;
        double acc_eps = 0.0;

        for (uint32_t base = 0; base < R; base += BA_NT) {
            __syncthreads();
            // ================= phase A: unrank supersequence base+tid of y', DP =================
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
                rc.info = miss0 | (miss1 << 1) | ((uint32_t)(t < 8 ? t : 8) << 8) | ((uint32_t)t << 16);
                rc.pad = 0u;
                s_rec[tid] = rc;
            }
            const int nn = (R - base < (uint32_t)BA_NT) ? (int)(R - base) : BA_NT;
            const int ngrp = (nn + BA_GRP - 1) / BA_GRP;
            __syncthreads();

            // ================= phase B =================
            auto issue_rows = [&](int g) {                     // stage the p rows of group g
                if (MODE != OUT_SWEEP) return;
                const int j = tid / (nv / 2 > 0 ? nv / 2 : 1);  // row of the group this thread copies a piece of
                const int piece = tid - j * (nv / 2);
                const int i = g * BA_GRP + j;
                if (j < BA_GRP && i < nn) {
                    const uint32_t dst = sStage + (uint32_t)((g & 1) * BA_GRP + j) * ROWB + (uint32_t)piece * 16u;
                    ba_cp_async16(dst, a.p + (((size_t)s_rec[i].id << m) + 2u * (size_t)piece));
                }
            };
            issue_rows(0);
            for (int g = 0; g < ngrp; g++) {
                ba_cp_async_wait_all();
                __syncthreads();
                if (g + 1 < ngrp) issue_rows(g + 1);

                // ---- the empty-z pair of every node: thread (v, node) ----------------------------------
                for (int e0 = 0; e0 < BA_GRP; e0 += epn) {
                    const int i = g * BA_GRP + e0 + esub;
                    if (esub < epn && e0 + esub < BA_GRP && i < nn) {
                        uint32_t al[9];
                        const uint4 r0 = *(const uint4 *)&s_rec[i].a[0], r1 = *(const uint4 *)&s_rec[i].a[4],
                                    r2 = *(const uint4 *)&s_rec[i].a[8];
                        al[0] = r0.x; al[1] = r0.y; al[2] = r0.z; al[3] = r0.w;
                        al[4] = r1.x; al[5] = r1.y; al[6] = r1.z; al[7] = r1.w; al[8] = r2.x;
                        const uint32_t u = r2.y, info = r2.z;
                        const int Lc = (int)((info >> 8) & 0xffu);
                        const uint32_t emb = ba_chain_single<4>(eW, 1u, evb, al, cy, Lc);
                        if (MODE == OUT_SWEEP) {
                            const uint32_t row = sStage + (uint32_t)((g & 1) * BA_GRP + e0 + esub) * ROWB;
                            acc_eps = fma(ba_u2d(emb), ba_lds_f64(row + (uint32_t)ev * 8u), acc_eps);
                        } else if (MODE == OUT_DEBUG) {
                            if (a.dbg_cz == 1u) a.dbg_out[((size_t)u << m) | (size_t)ev] = emb;
                        } else {
                            cnt_terms += 1ull; cnt_emb += emb;
                        }
                    }
                }
                // ---- pairs with a non-empty z: static z-major chunk schedule -------------------------------
                for (int j = 0; j < BA_GRP; j++) {
                    const int i = g * BA_GRP + j;
                    if (i >= nn) break;
                    const uint32_t info = s_rec[i].info;
                    const uint32_t mask = info & 3u;
                    if (!mask) continue;
                    uint32_t al[9];
                    const uint4 r0 = *(const uint4 *)&s_rec[i].a[0], r1 = *(const uint4 *)&s_rec[i].a[4],
                                r2 = *(const uint4 *)&s_rec[i].a[8];
                    al[0] = r0.x; al[1] = r0.y; al[2] = r0.z; al[3] = r0.w;
                    al[4] = r1.x; al[5] = r1.y; al[6] = r1.z; al[7] = r1.w; al[8] = r2.x;
                    const uint32_t u = r2.y;
                    const int Lc = (int)((info >> 8) & 0xffu);
                    const uint32_t sel1 = (cy & 1u) ? 0x4432u : 0x4410u;
                    const uint32_t row = sStage + (uint32_t)((g & 1) * BA_GRP + j) * ROWB;
#pragma unroll
                    for (int b = 0; b < 2; b++) {
                        if (!((mask >> b) & 1u)) continue;
#pragma unroll
                        for (int c = 0; c < BA_NC; c++) {
                            const uint2 d = dsc[b][c];
                            if (!__any_sync(0xffffffffu, d.x >> 31)) continue;
                            const uint32_t pa = sTz + (d.x & 0xfffffu);
                            uint32_t emb[BA_C], lk[BA_C], P[BA_C], vb[BA_C];
                            uint32_t anyl = 0u;
#pragma unroll
                            for (int q = 0; q < BA_C; q++) {
                                const uint2 wp = ba_lds_v2(pa + 8u * q);
                                P[q] = wp.y;
                                const uint32_t hw = __byte_perm(wp.x, 0u, sel1);
                                lk[q] = hw & 0xffu;
                                emb[q] = al[0] * (wp.y & 0xffu) + al[1] * (hw >> 8);   // al[s] = 0 beyond t
                                anyl |= lk[q];
                                vb[q] = sWv + (wp.y >> 16);
                            }
                            BaChain<2, BA_C, 4>::run(emb, lk, vb, anyl, al, cy, Lc);
                            if (MODE == OUT_SWEEP) {
#pragma unroll
                                for (int q = 0; q < BA_C; q++)
                                    acc[b][c] = fma(ba_u2d(emb[q]), ba_lds_f64(row + ((P[q] >> 5) & 0x7f8u)), acc[b][c]);
                            } else if (MODE == OUT_DEBUG) {
                                if ((d.x >> 31) && ((d.x >> 20) & 0x1ffu) == a.dbg_cz) {
#pragma unroll
                                    for (int q = 0; q < BA_C; q++)
                                        if (P[q] & 0xffu) a.dbg_out[((size_t)u << m) | (size_t)((P[q] >> 8) & 0xffu)] = emb[q];
                                }
                            } else {
#pragma unroll
                                for (int q = 0; q < BA_C; q++)
                                    if (P[q] & 0xffu) { cnt_terms += 1ull; cnt_emb += emb[q]; }
                            }
                        }
                    }
                }
            }
        }

        // ---- epilogue: fixed-order reduction of the chunks of each z, one write per (y', z) -----------------
        __syncthreads();                                       // records and rows are dead: the area becomes s_acc
        if (MODE == OUT_SWEEP) {
#pragma unroll
            for (int b = 0; b < 2; b++)
#pragma unroll
                for (int c = 0; c < BA_NC; c++) s_acc[((size_t)b * BA_NC + c) * BA_NT + tid] = acc[b][c];
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
            for (uint32_t zi = 1u + tid; zi < NZ; zi += BA_NT) {
                double s = 0.0;
                for (int q = s_csr_off[zi]; q < s_csr_off[zi + 1]; q++) s += s_acc[s_csr_idx[q]];
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
