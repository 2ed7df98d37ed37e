// ba_enum_in.cuh -- input sweep: for every x, enumerate its distinct subsequences y
// with their integer embedding counts emb(y,x) exactly once each.
//
// Work item = a high part u (h bits) with its 2^m inputs x = u.v; one persistent CTA per SM takes
// items from an atomic counter.  Per item:
//   phase A  every thread UNRANKS one node: the r-th distinct subsequence y' of u in trie pre-order
//            (the paper's stringUnrank idea, Alg. 4, with the subtree sizes Sub[pos] in the
//            role of the Count table P:260-274 and NextPos P:256-258 done with clz on bit masks), and
//            carries the integer embedding-count DP  E[i] = emb(y', u[0:i])  in registers along the
//            descent; the node record {alpha_0..8, code(y'), mask} goes to shared memory.
//   phase B  all threads walk the node list.  The (x,y) terms of a node are its pairs (v, z)
//            (ba_internal.h); they are dealt to the threads by a STATIC schedule: chunks of BA_C
//            consecutive entries of one v's list, the same chunks at every node, so each thread keeps
//            one FP64 accumulator per chunk in registers for the whole item and nothing is reduced or
//            synchronised per node.  emb(y'.z, u.v) is the integer chain sum_s alpha_s B(sigma_s.z, v)
//             walked through byte-packed prepend links; the operand c(y'.z) comes from the
//            node's row of c, staged with cp.async (9 contiguous segments of c, 16-byte pieces).
//   epilogue thread v adds the accumulators of v's chunks in a fixed order: D(x) = Hc(x) - sum_y emb c(y).
// MODE:
//   IN_SWEEP  D(x) and the fused reductions of 8(a3) (sum p D, max D, sum p 2^D per item)
//   IN_HC     Hc(x) = sum_y w_k emb log2(emb/ebar_k)   (iteration independent; built once per ctx)
//   IN_DEBUG  emb_out[idx(y)] = emb(y,x) for one x     (ba_debug_emb_row)
//   IN_COUNT  number of visited terms and sum of emb   (ba_debug_count_terms)
#pragma once
#include "ba_internal.h"

enum { IN_SWEEP = 0, IN_HC = 1, IN_DEBUG = 2, IN_COUNT = 3 };

struct InArgs {
    KConst kc;
    const uint2 *T64;         // v-major low table
    const uint32_t *vbase;    // [2^m]
    const uint2 *desc;        // [2][BA_NC][BA_NT]
    const uint16_t *csr_off;  // [2^m + 1]
    const uint16_t *csr_idx;
    int nT64, ncsr;
    const double *c;          // IN_SWEEP: c[code(y)], 2^{n+1} entries (entry 0 unused)
    const double *p;          // IN_SWEEP: p(x)
    double *Hc;               // IN_HC: out; IN_SWEEP: in
    double *D;                // IN_SWEEP: out
    double *part;             // IN_SWEEP: 3 doubles per u: sum p D, max D, sum p 2^D
    unsigned int *counter;    // work counter (zeroed before launch)
    uint32_t dbg_x;           // IN_DEBUG
    uint32_t *dbg_out;        // IN_DEBUG: NY zero-filled
    unsigned long long *cnt;  // IN_COUNT: [0] terms, [1] emb sum
};

struct InSmem { size_t T64, rec, ceps, stage, csr_off, csr_idx, sub, red, kcw, item, total; };

__host__ __device__ static inline InSmem enum_in_smem(int m, int nT64, int ncsr) {
    InSmem s;
    size_t o = 0;
    s.T64 = o; o += ((size_t)nT64 * 8 + 15) & ~(size_t)15;
    s.rec = o; o += (size_t)BA_NT * sizeof(NodeRec);
    s.ceps = o; o += (size_t)BA_NT * 8;
    s.stage = o;
    size_t st = (size_t)BA_NSTAGE * ((size_t)2 << m) * 8, ac = (size_t)2 * BA_NC * BA_NT * 8 + (size_t)BA_NT * 8;
    o += st > ac ? st : ac;                                // accumulator staging of the epilogue aliases the rows
    s.csr_off = o; o += (((size_t)(1 << m) + 1) * 2 + 15) & ~(size_t)15;
    s.csr_idx = o; o += ((size_t)ncsr * 2 + 15) & ~(size_t)15;
    s.sub = o; o += 32 * 4;
    s.red = o; o += 64 * 8;
    s.kcw = o; o += 2 * (BA_NMAX_I + 1) * 8;
    s.item = o; o += 16;
    s.total = o;
    return s;
}

template <int MODE>
__global__ void __launch_bounds__(BA_NT, 1) k_enum_in(const __grid_constant__ InArgs a) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int m = a.kc.m, h = a.kc.h, nv = 1 << m;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const InSmem L = enum_in_smem(m, a.nT64, a.ncsr);
    const uint32_t ROWB = (2u << m) * 8u;

    uint2 *s_T64 = (uint2 *)(smem + L.T64);
    NodeRec *s_rec = (NodeRec *)(smem + L.rec);
    double *s_ceps = (double *)(smem + L.ceps);
    double *s_stage = (double *)(smem + L.stage);
    double *s_acc = s_stage;                                // epilogue only
    uint16_t *s_csr_off = (uint16_t *)(smem + L.csr_off);
    uint16_t *s_csr_idx = (uint16_t *)(smem + L.csr_idx);
    uint32_t *s_sub = (uint32_t *)(smem + L.sub);
    double *s_red = (double *)(smem + L.red);
    double *s_w = (double *)(smem + L.kcw);
    double *s_lebar = s_w + (BA_NMAX_I + 1);
    uint32_t *s_item = (uint32_t *)(smem + L.item);

    for (int i = tid; i < a.nT64; i += BA_NT) s_T64[i] = a.T64[i];
    for (int i = tid; i <= nv; i += BA_NT) s_csr_off[i] = a.csr_off[i];
    for (int i = tid; i < a.ncsr; i += BA_NT) s_csr_idx[i] = a.csr_idx[i];
    for (int i = tid; i <= BA_NMAX_I; i += BA_NT) { s_w[i] = a.kc.w[i]; s_lebar[i] = a.kc.lebar[i]; }
    for (int i = tid; i < BA_NSTAGE; i += BA_NT) s_stage[(size_t)i * (ROWB / 8)] = 0.0;   // slot 0 of every row: padding pairs

    // static per-thread schedule
    uint2 dsc[2][BA_NC];
#pragma unroll
    for (int b = 0; b < 2; b++)
#pragma unroll
        for (int c = 0; c < BA_NC; c++) dsc[b][c] = a.desc[((size_t)b * BA_NC + c) * BA_NT + tid];
    const uint32_t sT64 = ba_smem_addr(s_T64);
    const uint32_t sStage = ba_smem_addr(s_stage);
    const int ev = tid & (nv - 1);                          // v of this thread's empty-z pair
    const int esub = tid >> m;                              // which node of an eps-round it serves
    const int epn = (BA_NT >> m) < BA_GRP ? (BA_NT >> m) : BA_GRP;   // nodes per eps-round
    const uint32_t evb = sT64 + a.vbase[ev] * 8u;           // v's list
    __syncthreads();
    const uint32_t eW = s_T64[a.vbase[ev] + 1].x;           // W of (v, empty)

    unsigned long long cnt_terms = 0, cnt_emb = 0;

    for (;;) {
        if (tid == 0) *s_item = (MODE == IN_DEBUG) ? (a.dbg_x >> m) : atomicAdd(a.counter, 1u);
        __syncthreads();
        const uint32_t u = *s_item;
        if (h < 32 && (u >> h) != 0) break;
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
        double acc_eps = 0.0;

        for (uint32_t base = 0; base < NN; base += BA_NT) {
            __syncthreads();                                   // previous chunk's records are no longer read
            // ================= phase A: unrank node base+tid, DP along the descent =================
            if (base + tid < NN) {
                uint32_t r = base + tid;
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
                const uint32_t miss0 = ba_nextpos(u, h, pos, 0u) >= h, miss1 = ba_nextpos(u, h, pos, 1u) >= h;
                NodeRec rc;
#pragma unroll
                for (int s = 0; s < 9; s++) rc.a[s] = al[s];
                rc.id = cy;
                rc.info = miss0 | (miss1 << 1) | ((uint32_t)(k < 8 ? k : 8) << 8) | ((uint32_t)k << 16);
                rc.pad = 0u;
                s_rec[tid] = rc;
                if (MODE == IN_SWEEP) s_ceps[tid] = a.c[cy];
            }
            const int nn = (NN - base < (uint32_t)BA_NT) ? (int)(NN - base) : BA_NT;
            const int ngrp = (nn + BA_GRP - 1) / BA_GRP;
            __syncthreads();

            // ================= phase B: pairs of every node =================
            auto issue_rows = [&](int g) {                     // stage the c rows of group g's masked nodes
                if (MODE != IN_SWEEP) return;
                if (tid >= nv) return;
#pragma unroll
                for (int j = 0; j < BA_GRP; j++) {
                    const int i = g * BA_GRP + j;
                    if (i >= nn) break;
                    if (!(s_rec[i].info & 3u)) continue;
                    const uint32_t cy = s_rec[i].id;
                    const uint32_t dst = sStage + (uint32_t)((g & 1) * BA_GRP + j) * ROWB;
                    if (tid == 0) {
                        ba_cp_async8(dst + 8u, a.c + cy);                              // row code 1: z empty
                    } else {
                        const uint32_t cz = 2u * tid;                                  // row codes cz, cz+1
                        const int jz = ba_len_of_code(cz);
                        ba_cp_async16(dst + cz * 8u, a.c + (((size_t)cy << jz) + (cz - (1u << jz))));
                    }
                }
            };
            issue_rows(0);
            for (int g = 0; g < ngrp; g++) {
                ba_cp_async_wait_all();
                __syncthreads();                               // rows of group g visible; group g-1 fully consumed
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
                        const uint32_t cy = r2.y, info = r2.z;
                        const int Lc = (int)((info >> 8) & 0xffu), k = (int)(info >> 16);
                        const uint32_t emb = ba_chain_single<8>(eW, 1u, evb, al, cy, Lc);
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
                    }
                }
                // ---- pairs with a non-empty z: static chunk schedule -------------------------------------
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
                    const uint32_t cy = r2.y;
                    const int Lc = (int)((info >> 8) & 0xffu), k = (int)(info >> 16);
                    const uint32_t sel1 = (cy & 1u) ? 0x4432u : 0x4410u;
                    const uint32_t row = sStage + (uint32_t)((g & 1) * BA_GRP + j) * ROWB;
#pragma unroll
                    for (int b = 0; b < 2; b++) {
                        if (!((mask >> b) & 1u)) continue;
#pragma unroll
                        for (int c = 0; c < BA_NC; c++) {
                            const uint2 d = dsc[b][c];
                            if (!__any_sync(0xffffffffu, d.x >> 31)) continue;
                            const uint32_t pa = sT64 + (d.x & 0xfffffu);
                            uint32_t emb[BA_C], lk[BA_C], P[BA_C], vb[BA_C];
                            uint32_t anyl = 0u;
#pragma unroll
                            for (int q = 0; q < BA_C; q++) {
                                const uint2 wp = ba_lds_v2(pa + 8u * q);
                                P[q] = wp.y;
                                const uint32_t hw = __byte_perm(wp.x, 0u, sel1);
                                lk[q] = hw & 0xffu;
                                emb[q] = al[0] * (wp.y & 0xffu) + al[1] * (hw >> 8);   // al[s] = 0 beyond k
                                anyl |= lk[q];
                                vb[q] = sT64 + d.y;
                            }
                            BaChain<2, BA_C, 8>::run(emb, lk, vb, anyl, al, cy, Lc);
                            if (MODE == IN_SWEEP) {
#pragma unroll
                                for (int q = 0; q < BA_C; q++)
                                    acc[b][c] = fma(ba_u2d(emb[q]), ba_lds_f64(row + (P[q] >> 16)), acc[b][c]);
                            } else if (MODE == IN_HC) {
#pragma unroll
                                for (int q = 0; q < BA_C; q++) {
                                    const int kk = k + (int)((P[q] >> 8) & 0xfu);
                                    const double wk = s_w[kk];
                                    if (wk != 0.0 && emb[q] > 0u) {
                                        const double le = (emb[q] > 1u) ? log2((double)emb[q]) : 0.0;
                                        acc[b][c] = fma(wk * (double)emb[q], le - s_lebar[kk], acc[b][c]);
                                    }
                                }
                            } else if (MODE == IN_DEBUG) {
                                const uint32_t v = (d.x >> 20) & 0xffu;
                                if ((d.x >> 31) && ((u << m) | v) == a.dbg_x) {
#pragma unroll
                                    for (int q = 0; q < BA_C; q++) {
                                        if (!(P[q] & 0xffu)) continue;
                                        const uint32_t cz = P[q] >> 19;
                                        const int jz = (int)((P[q] >> 8) & 0xfu);
                                        a.dbg_out[((size_t)cy << jz) + (cz - (1u << jz)) - 1u] = emb[q];
                                    }
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
                double S = 0.0;
                for (int t = ev; t < BA_NT; t += nv) S += s_acc[(size_t)2 * BA_NC * BA_NT + t];
                for (int q = s_csr_off[tid]; q < s_csr_off[tid + 1]; q++) S += s_acc[s_csr_idx[q]];
                const size_t x = ((size_t)u << m) | (size_t)tid;
                if (MODE == IN_HC) {
                    a.Hc[x] = S;
                } else {
                    const double Dx = a.Hc[x] - S;
                    a.D[x] = Dx;
                    const double px = a.p[x];
                    r0 = px * Dx; r1 = Dx; r2 = px * exp2(Dx);
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
            for (int i = tid; i < BA_NSTAGE; i += BA_NT) s_stage[(size_t)i * (ROWB / 8)] = 0.0;   // restore slot 0 of the rows
        }
        if (MODE == IN_DEBUG) break;
        __syncthreads();
    }
    if (MODE == IN_COUNT) {
        atomicAdd(&a.cnt[0], cnt_terms);
        atomicAdd(&a.cnt[1], cnt_emb);
    }
}
