// ba_enum_in.cuh -- input sweep: for every x, enumerate its distinct subsequences y
// with their integer embedding counts emb(y,x) exactly once each.
//
// One CTA owns a high part u (h bits) and its 2^m inputs x = u.v, thread v <-> input x (so D(x) is
// reduced in registers of one thread and written once: no atomics).  All warps walk the trie of
// distinct subsequences y' of u (the paper's NextPos walk, done with clz on bit masks)
// in lock step, each warp keeping its own copy of the embedding-count DP vectors
//     E[level][i] = emb(y', u[0:i])                       (the paper's O(nk) DP of P:173, one row per level)
// in shared memory.  A subsequence y of x = u.v is visited at the trie node y' that is its LONGEST
// prefix embeddable in u (y = y'.z, z empty or y'.z[0] not a subsequence of u), so each y is seen once.
// Its count follows from the concatenation identity P:181 with the low table (ba_internal.h):
//     emb(y'.z, u.v) = sum_{s>=0} emb(y'[0:k'-s], u) * emb(sigma_s.z, v),   sigma_s = last s symbols of y',
// where the first factor is the DFS stack of the trie walk and the second a chain of "prepend" links
// in v's list.  What is done with (y, emb) depends on MODE:
//   IN_SWEEP  D(x) = Hc(x) - sum_y emb(y,x) c(y), c(y) = w_k log2(A(y)/ebar_k) staged per y' in shared
//             memory from contiguous blocks of c (coalesced), plus the fused reductions of 8(a3)
//   IN_HC     Hc(x) = sum_y w_k emb log2(emb/ebar_k)   (iteration independent; built once per ctx)
//   IN_DEBUG  emb_out[idx(y)] = emb(y,x) for one x     (ba_debug_emb_row)
//   IN_COUNT  number of visited terms and sum of emb   (ba_debug_count_terms)
#pragma once
#include "ba_internal.h"

enum { IN_SWEEP = 0, IN_HC = 1, IN_DEBUG = 2, IN_COUNT = 3 };

struct InArgs {
    KConst kc;
    const uint32_t *tab;      // low table words
    const uint32_t *vinfo;    // per v
    int ntab;
    const double *c;          // IN_SWEEP: c(y), NY
    const double *p;          // IN_SWEEP: p(x)
    double *Hc;               // IN_HC: out; IN_SWEEP: in
    double *D;                // IN_SWEEP: out
    double *part;             // IN_SWEEP: 3 doubles per u: sum p D, max D, sum p 2^D
    unsigned int *counter;    // work counter (zeroed before launch)
    uint32_t dbg_x;           // IN_DEBUG
    uint32_t *dbg_out;        // IN_DEBUG: NY zero-filled
    unsigned long long *cnt;  // IN_COUNT: [0] terms, [1] emb sum
};

static inline size_t enum_in_smem_bytes(int m, int h, int ntab) {
    int nv = 1 << m, nwarp = (nv + 31) / 32, H1 = h + 1;
    size_t b = (size_t)ntab * 4 + (size_t)nv * 4;
    b = (b + 7) & ~(size_t)7;
    b += ((size_t)2 << m) * 8;                             // crow
    b += (size_t)nwarp * (H1 * H1 + 2 * H1) * 4;           // E, astk, pos per warp
    b = (b + 7) & ~(size_t)7;
    b += 64 * 8;                                           // reduction scratch
    b += 16;                                               // work item
    return b;
}

// emb(y'.z, u.v) by the prepend-link walk; astk[l] = emb(y'[0:l], u), kp = |y'|, cy = code(y').
__device__ __forceinline__ uint32_t ba_emb_walk(const uint32_t *tabv, uint32_t word,
                                                const uint32_t *astk, int kp, uint32_t cy) {
    uint32_t emb = astk[kp] * lt_B(word);
    uint32_t cur = word;
    for (int s = 0; s < kp; s++) {
        uint32_t l = lt_link(cur, (cy >> s) & 1u);
        if (l == BA_LINK_NONE) break;
        cur = tabv[l];
        emb += astk[kp - 1 - s] * lt_B(cur);
    }
    return emb;
}

template <int MODE>
__global__ void __launch_bounds__(256) k_enum_in(const __grid_constant__ InArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int m = a.kc.m, h = a.kc.h, nv = 1 << m, H1 = h + 1;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = (nv + 31) >> 5;
    const int nthr = blockDim.x;                 // max(32, 2^m); threads >= 2^m only take part in barriers
    const bool active = tid < nv;
    const uint32_t NZ = (2u << m) - 1u;

    uint32_t *s_tab = (uint32_t *)smem_raw;
    uint32_t *s_vinfo = s_tab + a.ntab;
    size_t off = ((size_t)(a.ntab + nv) * 4 + 7) & ~(size_t)7;
    double *s_crow = (double *)(smem_raw + off);
    off += ((size_t)2 << m) * 8;
    uint32_t *s_dfs = (uint32_t *)(smem_raw + off);
    off += (size_t)nwarp * (H1 * H1 + 2 * H1) * 4;
    off = (off + 7) & ~(size_t)7;
    double *s_red = (double *)(smem_raw + off);
    off += 64 * 8;
    uint32_t *s_item = (uint32_t *)(smem_raw + off);

    for (int i = tid; i < a.ntab; i += nthr) s_tab[i] = a.tab[i];
    for (int i = tid; i < nv; i += nthr) s_vinfo[i] = a.vinfo[i];
    __syncthreads();

    const uint32_t v = active ? tid : 0;
    const uint32_t vi = s_vinfo[v];
    const uint32_t *tabv = s_tab + vi_base(vi);
    const int n0 = vi_n0(vi), n1 = vi_n1(vi);

    uint32_t *E = s_dfs + (size_t)warp * (H1 * H1 + 2 * H1);
    uint32_t *astk = E + H1 * H1;
    uint32_t *pos = astk + H1;

    unsigned long long cnt_terms = 0, cnt_emb = 0;

    for (;;) {
        if (tid == 0) *s_item = (MODE == IN_DEBUG) ? (a.dbg_x >> m) : atomicAdd(a.counter, 1u);
        __syncthreads();
        const uint32_t u = *s_item;
        __syncthreads();
        if (h < 32 && (u >> h) != 0) break;
        if (MODE == IN_DEBUG && blockIdx.x != 0) break;

        double acc = 0.0;   // IN_SWEEP: sum emb c ; IN_HC: Hc

        // ---- trie walk over the distinct subsequences y' of u (all warps in lock step) -------------
        for (int i = lane; i <= h; i += 32) E[i] = 1u;      // emb(empty, u[0:i]) = 1
        if (lane == 0) { astk[0] = 1u; pos[0] = 0u; }
        __syncwarp();
        int level = 0;
        uint32_t cy = 1u;
        unsigned long long nc = 0ull;                         // 2 bits per level: next child to try
        bool visit = true;
        for (;;) {
            if (visit) {
                // ---------------- row y' = node at `level` ----------------
                const int kp = level;
                const int pl = (int)pos[level];
                const bool miss0 = ba_nextpos(u, h, pl, 0u) >= h;
                const bool miss1 = ba_nextpos(u, h, pl, 1u) >= h;
                const bool staged = (MODE == IN_SWEEP) && (miss0 || miss1);
                if (staged) {
                    __syncthreads();                           // readers of the previous row are done
                    for (uint32_t i = tid; i < NZ; i += nthr) {
                        const uint32_t cz = i + 1u;
                        const int j = ba_len_of_code(cz);
                        s_crow[i] = a.c[((size_t)cy << j) - 1u + (cz - (1u << j))];
                    }
                    __syncthreads();
                }
                double racc = 0.0;
                // entry ranges: [0,1) always; [1,1+n0) if 0 is missing after y' in u; [1+n0,1+n0+n1) if 1 is
                for (int blk = 0; blk < 3 && active; blk++) {
                    int e0, e1;
                    if (blk == 0) { e0 = 0; e1 = 1; }
                    else if (blk == 1) { if (!miss0) continue; e0 = 1; e1 = 1 + n0; }
                    else { if (!miss1) continue; e0 = 1 + n0; e1 = 1 + n0 + n1; }
                    for (int e = e0; e < e1; e++) {
                        const uint32_t word = tabv[e];
                        const uint32_t emb = ba_emb_walk(tabv, word, astk, kp, cy);
                        const uint32_t cz = lt_code(word);
                        if (MODE == IN_SWEEP) {
                            const double cv = staged ? s_crow[cz - 1u] : a.c[(size_t)cy - 1u];
                            racc = fma((double)emb, cv, racc);
                        } else if (MODE == IN_HC) {
                            const int k = kp + ba_len_of_code(cz);
                            const double wk = a.kc.w[k];
                            if (wk != 0.0) {
                                const double le = (emb > 1u) ? log2((double)emb) : 0.0;
                                racc = fma(wk * (double)emb, le - a.kc.lebar[k], racc);
                            }
                        } else if (MODE == IN_DEBUG) {
                            if (((u << m) | v) == a.dbg_x) {
                                const int j = ba_len_of_code(cz);
                                a.dbg_out[((size_t)cy << j) - 1u + (cz - (1u << j))] = emb;
                            }
                        } else {
                            cnt_terms += 1ull;
                            cnt_emb += emb;
                        }
                    }
                }
                acc += racc;
                visit = false;
                __syncwarp();                                  // lanes leave the row together (E/astk reuse)
            }
            const int ncl = (int)((nc >> (2 * level)) & 3ull);
            if (ncl < 2) {
                nc += (1ull << (2 * level));
                const uint32_t b = (uint32_t)ncl;
                const int pl = (int)pos[level];
                const int p = ba_nextpos(u, h, pl, b);
                if (p < h) {
                    const uint32_t *Ep = E + level * H1;
                    uint32_t *Ec = E + (level + 1) * H1;
                    uint32_t run = 0u;
                    for (int i = p; i < h; i++) {
                        if (((u >> (h - 1 - i)) & 1u) == b) run += Ep[i];
                        Ec[i + 1] = run;
                    }
                    level++;
                    pos[level] = (uint32_t)(p + 1);
                    astk[level] = run;
                    cy = (cy << 1) | b;
                    nc &= ~(3ull << (2 * level));
                    __syncwarp();
                    visit = true;
                }
            } else {
                if (level == 0) break;
                level--;
                cy >>= 1;
            }
        }

        // ---- epilogue: thread v owns x = u.v -------------------------------------------------------
        const size_t x = ((size_t)u << m) | v;
        if (MODE == IN_HC) {
            if (active) a.Hc[x] = acc;
        } else if (MODE == IN_SWEEP) {
            double r0 = 0.0, r1 = -INFINITY, r2 = 0.0;
            if (active) {
                const double Dx = a.Hc[x] - acc;
                a.D[x] = Dx;
                const double px = a.p[x];
                r0 = px * Dx; r1 = Dx; r2 = px * exp2(Dx);
            }
            for (int o = 16; o > 0; o >>= 1) {
                r0 += __shfl_xor_sync(0xffffffffu, r0, o);
                r1 = fmax(r1, __shfl_xor_sync(0xffffffffu, r1, o));
                r2 += __shfl_xor_sync(0xffffffffu, r2, o);
            }
            __syncthreads();
            if (lane == 0) { s_red[warp * 3] = r0; s_red[warp * 3 + 1] = r1; s_red[warp * 3 + 2] = r2; }
            __syncthreads();
            if (tid == 0) {
                double t0 = 0.0, t1 = -INFINITY, t2 = 0.0;
                for (int w = 0; w < nwarp; w++) {
                    t0 += s_red[w * 3];
                    t1 = fmax(t1, s_red[w * 3 + 1]);
                    t2 += s_red[w * 3 + 2];
                }
                a.part[(size_t)u * 3] = t0;
                a.part[(size_t)u * 3 + 1] = t1;
                a.part[(size_t)u * 3 + 2] = t2;
            }
        }
        if (MODE == IN_DEBUG) break;
        __syncthreads();
    }
    if (MODE == IN_COUNT) {
        atomicAdd(&a.cnt[0], cnt_terms);
        atomicAdd(&a.cnt[1], cnt_emb);
    }
}
