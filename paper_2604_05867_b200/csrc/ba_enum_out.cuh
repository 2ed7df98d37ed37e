// ba_enum_out.cuh -- output sweep: q(y) = w_k sum_{x contains y} emb(y,x) p(x) as a
// GATHER over the length-n supersequences of y: every output has a
// single owner, nothing is accumulated with atomics.
//
// Work item = a high output prefix y' (length t <= h, code cy).  The CTA that owns y' enumerates the
// length-h supersequences u of y' by unranking (the paper's subsetUnrank / RecSuperSeq, Alg. 5-6,
// P:471-563, with the G3 correction for the unmatched tail; their number is sum_{i<=h-t} C(h,i) by
// Lemma 6), computes for each u the integer counts alpha_s = emb(y'[0:t-s], u) with the
// textbook DP, and loads the 2^m consecutive inputs p(u.*) -- the run of inputs whose low m bits are
// free (SURVEY 7.2 "coalescing the gather") -- into shared memory with one coalesced row load.
// Each (x = u.v, y = y'.z) term is visited exactly once, at the item y' that is the longest prefix of
// y embeddable in u (z empty or y'.z[0] not in u after the greedy match), with
//     emb(y'.z, u.v) = sum_s alpha_s * emb(sigma_s.z, v)            (low table, ba_internal.h)
// The CTA owns the partial sums Apart[y'][z] for all z in {0,1}^{<=m}; thread groups of 2^{m-j}
// threads share one z of length j and split its supersequences v (Lemma 6 makes every z of one length
// equally expensive).  k_out_final then adds, in a fixed order, the <= m+1 partials of each y:
//     A(y) = sum_j Apart[y[0:k-j]][y[k-j:]],   q(y) = w_k A(y),   c(y) = w_k log2(A(y)/ebar_k).
#pragma once
#include "ba_internal.h"

enum { OUT_SWEEP = 0, OUT_DEBUG = 1, OUT_COUNT = 2 };

#define BA_OUT_RB 8     // p-rows staged per barrier pair

__constant__ uint32_t c_binom[BA_NMAX_I + 1][BA_NMAX_I + 1];

struct OutArgs {
    KConst kc;
    OutLayout lay;
    const uint32_t *tab;
    const uint32_t *vinfo;
    const uint16_t *thrlist;   // [total slots][2^m]
    int ntab;
    const double *p;           // NX
    double *Apart;             // (2^{h+1}-1) * (2^{m+1}-1)
    unsigned int *counter;
    uint32_t dbg_cy;           // OUT_DEBUG: code of the target y
    uint32_t *dbg_out;         // OUT_DEBUG: NX zero-filled
    unsigned long long *cnt;   // OUT_COUNT
};

static inline size_t enum_out_smem_bytes(int m, int ntab, int total_slots) {
    int nv = 1 << m, nthr = nv < 32 ? 32 : nv;
    size_t b = (size_t)ntab * 4 + (size_t)nv * 4;
    b += (size_t)total_slots * nv * 2;
    b = (b + 7) & ~(size_t)7;
    b += (size_t)BA_OUT_RB * nv * 8;                 // p rows
    b += (size_t)nthr * 8;                           // reduction scratch
    b += (size_t)nthr * (4 + 4 + 4 * (BA_MLOW + 1)); // row records: u, mask, alpha[m+1]
    b += 16;
    return b;
}

// emb(y'.z, u.v): alpha[s] = emb(y'[0:t-s], u) for s <= min(t,m)
__device__ __forceinline__ uint32_t ba_emb_walk_out(const uint32_t *tabv, uint32_t word,
                                                    const uint32_t *alpha, int t, uint32_t cy) {
    uint32_t emb = alpha[0] * lt_B(word);
    uint32_t cur = word;
    for (int s = 0; s < t; s++) {
        uint32_t l = lt_link(cur, (cy >> s) & 1u);
        if (l == BA_LINK_NONE) break;
        cur = tabv[l];
        emb += alpha[s + 1] * lt_B(cur);
    }
    return emb;
}

template <int MODE>
__global__ void __launch_bounds__(256) k_enum_out(const __grid_constant__ OutArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int m = a.kc.m, h = a.kc.h, nv = 1 << m;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const bool active = tid < nv;
    const uint32_t NZ = (2u << m) - 1u;
    const int total_slots = a.lay.off[m + 1];

    uint32_t *s_tab = (uint32_t *)smem_raw;
    uint32_t *s_vinfo = s_tab + a.ntab;
    uint16_t *s_tl = (uint16_t *)(s_vinfo + nv);
    size_t off = ((size_t)(a.ntab + nv) * 4 + (size_t)total_slots * nv * 2 + 7) & ~(size_t)7;
    double *s_prow = (double *)(smem_raw + off);
    off += (size_t)BA_OUT_RB * nv * 8;
    double *s_red = (double *)(smem_raw + off);
    off += (size_t)nthr * 8;
    uint32_t *s_ru = (uint32_t *)(smem_raw + off);
    uint32_t *s_rmask = s_ru + nthr;
    uint32_t *s_ralpha = s_rmask + nthr;               // [nthr][m+1]
    off += (size_t)nthr * (4 + 4 + 4 * (BA_MLOW + 1));
    uint32_t *s_item = (uint32_t *)(smem_raw + off);

    for (int i = tid; i < a.ntab; i += nthr) s_tab[i] = a.tab[i];
    for (int i = tid; i < nv; i += nthr) s_vinfo[i] = a.vinfo[i];
    for (int i = tid; i < total_slots * nv; i += nthr) s_tl[i] = a.thrlist[i];
    __syncthreads();

    const uint32_t my_v = active ? tid : 0;
    const uint32_t *my_tabv = s_tab + vi_base(s_vinfo[my_v]);
    const uint32_t topbit = (m > 0) ? ((my_v >> (m - 1)) & 1u) : 0u;   // z[0] of every z (|z|>=1) this thread serves

    unsigned long long cnt_terms = 0, cnt_emb = 0;
    const uint32_t n_items = (h >= 31) ? 0xffffffffu : ((2u << h) - 1u);   // codes 1 .. 2^{h+1}-1

    for (uint32_t dbg_j = 0;; dbg_j++) {
        uint32_t cy;
        if (MODE == OUT_DEBUG) {
            // the splits y = y'.z of the target: |z| = j, y' = y >> j
            const int ky = ba_len_of_code(a.dbg_cy);
            if ((int)dbg_j > m || (int)dbg_j > ky) break;
            if (ky - (int)dbg_j > h) continue;
            cy = a.dbg_cy >> dbg_j;
        } else {
            if (tid == 0) *s_item = atomicAdd(a.counter, 1u);
            __syncthreads();
            cy = *s_item + 1u;
            __syncthreads();
            if (cy > n_items) break;
        }
        const int t = ba_len_of_code(cy);
        const uint32_t yv = cy - (1u << t);
        // number of supersequences of y' of length h: sum_{w <= h-t} C(h,w)   (Lemma 6)
        uint32_t R = 0;
        for (int w = 0; w <= h - t; w++) R += c_binom[h][w];

        double acc[BA_MLOW + 1];
#pragma unroll
        for (int j = 0; j <= BA_MLOW; j++) acc[j] = 0.0;

        for (uint32_t b0 = 0; b0 < R; b0 += nthr) {
            // ---- each thread unranks one supersequence u of y' and runs the count DP ----------------
            const uint32_t ri = b0 + tid;
            if (ri < R) {
                uint32_t w = 0, rem = ri;
                while (rem >= c_binom[h][w]) { rem -= c_binom[h][w]; w++; }
                // subsetUnrank(h, w, rem): S = positions not used by the greedy match (Alg. 5)
                uint32_t S = 0;
                {
                    uint32_t ww = w, j = rem;
                    for (int pp = 0; pp < h && ww > 0; pp++) {
                        const uint32_t cc = c_binom[h - pp - 1][ww - 1];
                        if (j < cc) { S |= 1u << pp; ww--; } else { j -= cc; }
                    }
                }
                // RecSuperSeq (Alg. 6 with G3): build u left to right
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
                // alpha_s = emb(y'[0:t-s], u): textbook DP over the positions of u
                uint32_t e[BA_NMAX_I + 1];
                e[0] = 1u;
                for (int rr = 1; rr <= t; rr++) e[rr] = 0u;
                for (int pp = 0; pp < h; pp++) {
                    const uint32_t ub = (u >> (h - 1 - pp)) & 1u;
                    const int top = (pp + 1 < t) ? pp + 1 : t;
                    for (int rr = top; rr >= 1; rr--)
                        if (((yv >> (t - rr)) & 1u) == ub) e[rr] += e[rr - 1];
                }
                s_ru[tid] = u;
                const uint32_t miss0 = ba_nextpos(u, h, ell, 0u) >= h;
                const uint32_t miss1 = ba_nextpos(u, h, ell, 1u) >= h;
                s_rmask[tid] = miss0 | (miss1 << 1);
                for (int s = 0; s <= m; s++) s_ralpha[tid * (BA_MLOW + 1) + s] = (s <= t) ? e[t - s] : 0u;
            }
            __syncthreads();
            const uint32_t nb = (R - b0 < (uint32_t)nthr) ? (R - b0) : (uint32_t)nthr;
            for (uint32_t r0 = 0; r0 < nb; r0 += BA_OUT_RB) {
                const uint32_t nr = (nb - r0 < BA_OUT_RB) ? (nb - r0) : BA_OUT_RB;
                if (MODE != OUT_COUNT && MODE != OUT_DEBUG) {
                    if (active)
                        for (uint32_t rr = 0; rr < nr; rr++)
                            s_prow[rr * nv + tid] = a.p[((size_t)s_ru[r0 + rr] << m) | tid];
                    __syncthreads();
                }
                for (uint32_t rr = 0; rr < nr && active; rr++) {
                    const uint32_t row = r0 + rr;
                    const uint32_t *alpha = s_ralpha + row * (BA_MLOW + 1);
                    const uint32_t mask = s_rmask[row];
                    const double *prow = s_prow + rr * nv;
                    const uint32_t u = s_ru[row];
                    // class 0: z = empty, v = my_v
                    {
                        const uint32_t emb = ba_emb_walk_out(my_tabv, my_tabv[0], alpha, t, cy);
                        if (MODE == OUT_SWEEP) acc[0] = fma((double)emb, prow[my_v], acc[0]);
                        else if (MODE == OUT_COUNT) { cnt_terms++; cnt_emb += emb; }
                        else if (dbg_j == 0) a.dbg_out[((size_t)u << m) | my_v] = emb;
                    }
                    if (!((mask >> topbit) & 1u)) continue;
#pragma unroll
                    for (int j = 1; j <= BA_MLOW; j++) {
                        if (j > m) break;
                        if (MODE == OUT_DEBUG) {
                            // only the group that serves the target's z of length dbg_j
                            if (j != (int)dbg_j) continue;
                            if ((my_v >> (m - j)) != (a.dbg_cy & ((1u << j) - 1u))) continue;
                        }
                        const int s0 = a.lay.off[j], s1 = a.lay.off[j + 1];
                        double aj = 0.0;
                        for (int sl = s0; sl < s1; sl++) {
                            const uint32_t ent = s_tl[sl * nv + tid];
                            if (!tl_valid(ent)) continue;
                            const uint32_t v = tl_v(ent);
                            const uint32_t *tabv = s_tab + vi_base(s_vinfo[v]);
                            const uint32_t emb = ba_emb_walk_out(tabv, tabv[tl_el(ent)], alpha, t, cy);
                            if (MODE == OUT_SWEEP) aj = fma((double)emb, prow[v], aj);
                            else if (MODE == OUT_COUNT) { cnt_terms++; cnt_emb += emb; }
                            else a.dbg_out[((size_t)u << m) | v] = emb;
                        }
                        acc[j] += aj;
                    }
                }
                if (MODE != OUT_COUNT && MODE != OUT_DEBUG) __syncthreads();
            }
            __syncthreads();
        }

        // ---- owner-side reduction of the thread groups, fixed order, and the single write -----------
        if (MODE == OUT_SWEEP) {
#pragma unroll
            for (int j = 0; j <= BA_MLOW; j++) {
                if (j > m) break;
                s_red[tid] = acc[j];
                __syncthreads();
                const int G = 1 << (m - j);
                if (active && (tid & (G - 1)) == 0) {
                    double sum = 0.0;
                    for (int g = 0; g < G; g++) sum += s_red[tid + g];
                    a.Apart[(size_t)(cy - 1u) * NZ + ((1u << j) - 1u) + (tid >> (m - j))] = sum;
                }
                __syncthreads();
            }
        }
    }
    if (MODE == OUT_COUNT) {
        atomicAdd(&a.cnt[0], cnt_terms);
        atomicAdd(&a.cnt[1], cnt_emb);
    }
}
