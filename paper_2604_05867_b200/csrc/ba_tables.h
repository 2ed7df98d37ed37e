// ba_tables.h -- host-side construction of the static low tables and pair schedules of the ENUM
// kernels (formats: ba_internal.h).  Everything here depends on m = min(n, 8) only.
#pragma once
#include "ba_internal.h"

#include <algorithm>
#include <utility>
#include <vector>

// One side (input sweep or output sweep) of the pair schedule, see ba_internal.h "GROUPS".
struct GroupSide {
    std::vector<uint4> GB;          // [BA_NCLS][2][BA_KG][BA_NT]: B_0 | B_1<<8 | B_2<<16 | B_3<<24 of the group's 4 slots
    std::vector<uint32_t> GA;       // [2][BA_KG][BA_NT]: byte offset of the group's operand in a staged row
    std::vector<uint16_t> GO;       // [2][BA_KG][BA_GP][BA_NT]: owner of the slot (in: v, out: code(z)); 0xffff = unused
    std::vector<uint16_t> GW;       // [2][BA_NT/32]: half 0 | half 1 << 8; a half = groups in use (0..2) | loop type << 2 (1: only B_0 ever; 2: B_2 = B_3 = 0 always; 4)
    std::vector<uint16_t> csr_off;  // [2][nown + 1]: slots of an owner, per list
    std::vector<uint16_t> csr_idx;  // [2][BA_KG*BA_GP*BA_NT]: slot index (k*BA_GP + q)*BA_NT + tid
    int nown = 0;                   // in: 2^m ; out: 2^{m+1} (by code(z))
    int nsc = 1;                    // schedules: 2 (input sweep: by the last symbol of y') or BA_NCLS (output sweep: by class)
    std::vector<uint4> R;           // riders [BA_NCLS][2][nr]: {B0..B3, B4 | owner << 16, row byte offset, 0}, sorted by owner
    std::vector<uint16_t> r_cnt;    // [BA_NCLS][2]
    std::vector<uint16_t> r_csr;    // [BA_NCLS][2][nown + 1] rider range of an owner
    std::vector<uint32_t> R8;       // [BA_NCLS][2][8][nr]: bytes = B_4..B_7 of the rider for sigma bits 4..6 (B_7 reads 7 symbols of sigma; B_8 = 0)
    int nr = 0;
    unsigned long long npairs[2] = {0, 0}, nslots[2] = {0, 0}, ngroups[2] = {0, 0};   // statistics
};

struct TileTables {
    int m = 0, nv = 0;
    GroupSide in, out;
    GroupSide inf;                  // input sweep, IN_SWEEP: every pair keeps its slot with B_0..B_3 under every class and there are
                                    // no riders -- the deep part of the chains (s >= 4) is summed in factored form by the kernel
    std::vector<uint2> EPS8;        // [256][nv]: byte s = B(sigma_s, v), s = 0..7, sigma = the row index
    std::vector<uint32_t> EPSH;     // [BA_NCLS][8][nv]: EPS8[(hi << 4) | cls][v].y, hi = sigma bits 4..6: the slice of a class (input sweep)
    std::vector<uint8_t> LT;        // [nv][2^{m+1}]: emb(w, v) by code(w) (entry 0 unused): the whole low tile (k_low_tile)
    std::vector<uint32_t> LTV_off;  // [nv + 1]: the subsequences w of v (the empty one included) ...
    std::vector<uint32_t> LTV;      // ... as code(w) << 8 | emb(w, v), by increasing code (input sweep: pairs (v, empty))
    bool ok = false;
};

// code of sigma_s . z, sigma_s = low s bits of sig (the last s symbols of y')
static inline uint32_t tt_prepend(uint32_t sig, int s, uint32_t cz) {
    const int lz = 31 - __builtin_clz(cz);
    return (1u << (lz + s)) | ((sig & ((1u << s) - 1u)) << lz) | (cz - (1u << lz));
}

struct TTPair { int v; uint32_t cz; };
#ifndef BA_G2_EXTRA
#define BA_G2_EXTRA 3.0                     // instructions per node a warp that sums the deep part spends on it
#endif
#ifndef BA_STAGER_EXTRA
#define BA_STAGER_EXTRA 12.0                // instructions per node the stager warp spends on staging (measured best of 0 / 12 / 25)
#endif

// Deal the pairs of one list to (warp, level, lane, slot):
//   * a GROUP is up to BA_GP pairs that share their gathered operand (`key` = its position in a staged row); the
//     thread fetches the operand once per node and uses it for the group's pairs;
//   * groups are of TYPE 2 (no pair of the group ever has B_2 != 0 in a fast slot: one dot-product instruction per
//     term) or 4; 32 groups of one type, consecutive in operand order, form a LEVEL (one group per lane: their operand
//     fetch reads neighbouring or equal row positions); a warp carries up to BA_KG levels of ONE type, so that the
//     node loop is straight-line code chosen per warp;
//   * warps are filled so that the four schedulers of the SM carry about the same number of instructions.
template <typename KeyOf, typename OwnerOf, typename BPack, typename DeepOf>
static bool tt_deal(int m, int b, int sc, uint32_t clsmask, const std::vector<TTPair> &pairs, KeyOf key_of, OwnerOf owner_of,
                    BPack bpack, DeepOf deep, const double *warp_extra, GroupSide &S) {
    // sc = schedule index; clsmask = the classes it serves.  Output sweep: one schedule per class (an item has one
    // class, so its slots are typed and filled for that class alone).  Input sweep: one schedule per LAST SYMBOL of y'
    // (class bit 0): whether a pair can have B_1 at all depends on that symbol only, and the kernel switches its
    // accumulators between the two schedules once per super-batch.
    struct Grp { int type; uint32_t key; std::vector<int> items; };
    const int np = (int)pairs.size();
    std::vector<int> ptype(np, 1);
    for (int i = 0; i < np; i++)
        for (int cls = 0; cls < BA_NCLS; cls++) {
            if (!((clsmask >> cls) & 1u) || deep(cls, pairs[i])) continue;
            const uint32_t bp = bpack(cls, pairs[i]);
            if ((bp >> 16) && ptype[i] < 4) ptype[i] = 4;
            else if ((bp >> 8) && ptype[i] < 2) ptype[i] = 2;
        }
    // ---- groups per operand: type-4 pairs first, the type-2 pairs fill up the last type-4 group
    std::vector<std::vector<int>> by_key(2u << m);
    for (int i = 0; i < np; i++) by_key[key_of(pairs[i])].push_back(i);
    std::vector<Grp> groups;
    for (uint32_t k = 0; k < by_key.size(); k++) {
        std::vector<int> &L = by_key[k];
        if (L.empty()) continue;
        std::stable_sort(L.begin(), L.end(), [&](int x, int y) { return ptype[x] > ptype[y]; });
        for (size_t i = 0; i < L.size(); i += BA_GP) {
            Grp g;
            g.key = k;
            g.type = ptype[L[i]];
            for (size_t j = i; j < L.size() && j < i + BA_GP; j++) g.items.push_back(L[j]);
            groups.push_back(g);
        }
    }
    std::stable_sort(groups.begin(), groups.end(), [](const Grp &x, const Grp &y) { return x.type != y.type ? x.type > y.type : x.key < y.key; });
    // ---- levels of 32 groups of one type
    struct Lvl { int type; std::vector<int> g; };
    std::vector<Lvl> levels;
    for (size_t i = 0; i < groups.size(); i++) {
        if (levels.empty() || levels.back().type != groups[i].type || levels.back().g.size() == 32) levels.push_back(Lvl{groups[i].type, {}});
        levels.back().g.push_back((int)i);
    }
    const int NW = BA_NT / 32;
    // ---- HALVES: up to 2 levels of one type; a warp carries two halves (ba_internal.h "ba_half_loop").  Cost of a level
    // in instructions per node and lane: type 4: 4 x (2 IDP + MOV + DADD + DFMA), type 2: 4 x 4, type 1: 4 DFMA + DMUL + LDS.
    struct Half { int type; std::vector<int> lv; double cost; };
    auto cost_of = [](int type) { return type == 4 ? 20.5 : type == 2 ? 16.5 : 6.5; };
    std::vector<Half> halves;
    for (size_t i = 0; i < levels.size();) {
        Half hf; hf.type = levels[i].type;
        hf.lv.push_back((int)i);
        if (i + 1 < levels.size() && levels[i + 1].type == hf.type) hf.lv.push_back((int)i + 1);
        hf.cost = cost_of(hf.type) * hf.lv.size() + 1.5;
        i += hf.lv.size();
        halves.push_back(hf);
    }
    if ((int)halves.size() > 2 * NW) return false;
    // free half slots: split the heaviest two-level halves, so that the warps can be levelled better
    while ((int)halves.size() < 2 * NW) {
        int best = -1;
        for (size_t i = 0; i < halves.size(); i++)
            if (halves[i].lv.size() == 2 && (best < 0 || halves[i].cost > halves[best].cost)) best = (int)i;
        if (best < 0) break;
        Half nh; nh.type = halves[best].type; nh.lv.push_back(halves[best].lv[1]); nh.cost = cost_of(nh.type) + 1.5;
        halves[best].lv.pop_back(); halves[best].cost = nh.cost;
        halves.push_back(nh);
    }
    // ---- halves -> warps: heaviest first onto the warp with the least load that has a free half; warp_extra[w] =
    // instructions per node the warp spends outside its levels (riders); ties go to the scheduler (warp & 3) with the
    // least load
    std::stable_sort(halves.begin(), halves.end(), [](const Half &x, const Half &y) { return x.cost > y.cost; });
    double wload[BA_NT / 32], sload[4] = {0, 0, 0, 0};
    int nh_of[BA_NT / 32];
    for (int w = 0; w < NW; w++) { wload[w] = warp_extra[w]; nh_of[w] = 0; sload[w & 3] += warp_extra[w]; }
    for (auto &hf : halves) {
        int warp = -1;
        for (int w = 0; w < NW; w++) {
            if (nh_of[w] >= 2) continue;
            if (warp < 0 || wload[w] < wload[warp] - 1e-9 || (wload[w] < wload[warp] + 1e-9 && sload[w & 3] < sload[warp & 3] - 1e-9)) warp = w;
        }
        if (warp < 0) return false;
        const int hslot = nh_of[warp]++;
        wload[warp] += hf.cost; sload[warp & 3] += hf.cost;
        S.GW[((size_t)sc * 2 + b) * NW + warp] |= (uint16_t)(((int)hf.lv.size() | (hf.type << 2)) << (8 * hslot));
        for (size_t kk = 0; kk < hf.lv.size(); kk++) {
            const int k = 2 * hslot + (int)kk;
            const Lvl &lv = levels[hf.lv[kk]];
            for (size_t l = 0; l < lv.g.size(); l++) {
                const Grp &g = groups[lv.g[l]];
                const int tid = warp * 32 + (int)l;
                S.GA[(((size_t)sc * 2 + b) * BA_KG + k) * BA_NT + tid] = 8u * g.key;
                for (size_t q = 0; q < g.items.size(); q++) {
                    const TTPair &pr = pairs[g.items[q]];
                    S.GO[((((size_t)sc * 2 + b) * BA_KG + k) * BA_GP + q) * BA_NT + tid] = (uint16_t)owner_of(pr);
                    for (int cls = 0; cls < BA_NCLS; cls++) {
                        if (!((clsmask >> cls) & 1u) || deep(cls, pr)) continue;                   // served by a rider under this class
                        uint4 &e = S.GB[(((size_t)cls * 2 + b) * BA_KG + k) * BA_NT + tid];
                        const uint32_t bp = bpack(cls, pr);
                        (q == 0 ? e.x : q == 1 ? e.y : q == 2 ? e.z : e.w) = bp;
                    }
                }
                S.nslots[b] += BA_GP;
            }
        }
    }
    S.npairs[b] += (unsigned long long)np;
    S.ngroups[b] += groups.size();
    return true;
}

static inline void build_tile_tables(int m, TileTables &T) {
    const int nv = 1 << m, NZc = 2 << m;                   // string codes 1 .. NZc-1
    T.m = m; T.nv = nv; T.ok = false;
    // ---- B[code(w)][v] = emb(w, v): textbook DP over the positions of v, all prefixes of w at once ------
    std::vector<uint8_t> B((size_t)NZc * nv, 0);
    for (int v = 0; v < nv; v++)
        for (int lw = 0; lw <= m; lw++)
            for (uint32_t w = 0; w < (1u << lw); w++) {
                uint32_t e[BA_MLOW + 2];
                for (int r = 0; r <= lw; r++) e[r] = (r == 0);
                for (int i = 0; i < m; i++) {
                    const uint32_t vb = ((uint32_t)v >> (m - 1 - i)) & 1u;
                    for (int r = lw; r >= 1; r--)
                        if (((w >> (lw - r)) & 1u) == vb) e[r] += e[r - 1];
                }
                B[(size_t)((1u << lw) | w) * nv + v] = (uint8_t)e[lw];       // <= C(8,4) = 70
            }
    T.LT.assign((size_t)nv * NZc, 0);
    for (int v = 0; v < nv; v++)
        for (int cw = 1; cw < NZc; cw++) T.LT[(size_t)v * NZc + cw] = B[(size_t)cw * nv + v];
    T.LTV_off.assign((size_t)nv + 1, 0u);
    T.LTV.clear();
    for (int v = 0; v < nv; v++) {
        for (int cw = 1; cw < NZc; cw++)
            if (B[(size_t)cw * nv + v]) T.LTV.push_back(((uint32_t)cw << 8) | B[(size_t)cw * nv + v]);
        T.LTV_off[v + 1] = (uint32_t)T.LTV.size();
    }
    auto Bof = [&](uint32_t cw, int v) -> uint32_t { return (cw < (uint32_t)NZc) ? B[(size_t)cw * nv + v] : 0u; };
    auto first_bit = [](uint32_t cz) -> int { const int lz = 31 - __builtin_clz(cz); return (int)((cz >> (lz - 1)) & 1u); };
    auto deep = [&](int cls, const TTPair &p) -> bool {        // chain of (v,z) under class cls reaches s = BA_KB
        const int lz = 31 - __builtin_clz(p.cz);
        return lz + BA_KB <= m && Bof(tt_prepend((uint32_t)cls, BA_KB, p.cz), p.v) != 0;
    };
    auto tail_of = [](uint32_t cz) -> uint32_t {               // code(t) for z = b.t
        const int lz = 31 - __builtin_clz(cz);
        return (1u << (lz - 1)) | (cz & ((1u << (lz - 1)) - 1u));
    };
    auto bpack = [&](int cls, const TTPair &p) -> uint32_t {   // B_0..B_3 under class cls
        uint32_t x = 0;
        const int lz = 31 - __builtin_clz(p.cz);
        for (int s = 0; s < 4; s++)
            if (lz + s <= m) x |= Bof(tt_prepend((uint32_t)cls, s, p.cz), p.v) << (8 * s);
        return x;
    };

    const int NW = BA_NT / 32;
    auto init_side = [&](GroupSide &S, int nown, int nsc) {
        S.nown = nown; S.nsc = nsc;
        S.GB.assign((size_t)BA_NCLS * 2 * BA_KG * BA_NT, make_uint4(0u, 0u, 0u, 0u));
        S.GA.assign((size_t)nsc * 2 * BA_KG * BA_NT, 0u);
        S.GO.assign((size_t)nsc * 2 * BA_KG * BA_GP * BA_NT, 0xffffu);
        S.GW.assign((size_t)nsc * 2 * NW, 0);
        S.csr_off.assign((size_t)nsc * 2 * (nown + 1), 0);
        S.csr_idx.assign((size_t)nsc * 2 * BA_KG * BA_GP * BA_NT, 0);
    };
    init_side(T.in, nv, 2);
    init_side(T.out, NZc, BA_NCLS);
    init_side(T.inf, nv, 2);
    auto deep_real = deep;

    for (int sidx = 0; sidx < 3; sidx++) {
        const int side = sidx & 1;
        const bool fact = (sidx == 2);                         // the factored-deep variant of the input side: no pair is left to a rider
        GroupSide &S = (sidx == 1) ? T.out : (sidx == 2) ? T.inf : T.in;
        auto deep = [&](int cls, const TTPair &p) -> bool { return fact ? false : deep_real(cls, p); };
        // operand position in a staged row.  in: the operand of z = b.t is c(y'.b.t) at position code(t) of the
        // node's half row; out: the operand of (v, z) is p(u.v) at position v of the node's row.
        // (the one-symbol z = "b" sits at position b, not 1: the staged half row starts with the 16-byte pair
        // c(y'.0), c(y'.1), so that every piece of it is a bulk copy)
        auto key_of = [&](const TTPair &p) -> uint32_t {
            if (side) return (uint32_t)p.v;
            const uint32_t tc = tail_of(p.cz);
            return tc == 1u ? (uint32_t)(p.cz & 1u) : tc;
        };
        auto owner_of = [&](const TTPair &p) -> uint32_t { return side ? p.cz : (uint32_t)p.v; };
        std::vector<std::vector<uint4>> riders((size_t)BA_NCLS * 2);
        std::vector<std::vector<TTPair>> rider_pairs((size_t)BA_NCLS * 2);
        S.r_csr.assign((size_t)BA_NCLS * 2 * (S.nown + 1), 0);
        for (int b = 0; b < 2; b++) {
            std::vector<TTPair> pairs;
            for (int v = 0; v < nv; v++)
                for (uint32_t cz = 2; cz < (uint32_t)NZc; cz++)
                    if (Bof(cz, v) && first_bit(cz) == b) pairs.push_back(TTPair{v, cz});
            // riders (the pairs deep under the class) sit on fixed threads: input sweep, two replicas on the last warps
            // of each half of the CTA, every other node each; output sweep, the last warps
            size_t ndeep = 0;
            for (int cls = 0; cls < BA_NCLS; cls++) {
                size_t c = 0;
                for (const TTPair &p : pairs) c += deep(cls, p);
                ndeep = std::max(ndeep, c);
            }
            double warp_extra[BA_NT / 32];
            const int rw = (int)((ndeep + 31) / 32);
            for (int w = 0; w < NW; w++)
                warp_extra[w] = side ? (w >= NW - rw ? 14.0 : 0.0) : ((w & (NW / 2 - 1)) >= NW / 2 - rw ? 8.0 : 0.0);
            if (fact)                                          // in: the warps that sum the deep part (BA_G2_NT targets, two replicas)
                for (int w = 0; w < NW; w++) warp_extra[w] = (!side && (w & (NW / 2 - 1)) >= NW / 2 - (BA_G2_NT + 31) / 32) ? BA_G2_EXTRA : 0.0;
            warp_extra[0] += BA_STAGER_EXTRA;                  // warp 0 also stages the batches: it must run ahead, not behind
            for (int sc = 0; sc < S.nsc; sc++) {
                // input sweep: schedule sc serves the classes with bit 0 = sc; output sweep: class sc
                const uint32_t clsmask = (S.nsc == BA_NCLS) ? (1u << sc) : (S.nsc == 2) ? (0x5555u << sc) : 0xffffu;
                std::vector<TTPair> sp;                        // a per-class schedule leaves the class's deep pairs to the riders
                for (const TTPair &p : pairs)
                    if (S.nsc != BA_NCLS || !deep(sc, p)) sp.push_back(p);
                if (!tt_deal(m, b, sc, clsmask, sp, key_of, owner_of, bpack, deep, warp_extra, S)) return;
                // ---- CSR of the epilogue: the slots of every owner, in slot order
                const size_t sb = (size_t)sc * 2 + b;
                std::vector<std::vector<uint16_t>> slots(S.nown);
                for (int k = 0; k < BA_KG; k++)
                    for (int q = 0; q < BA_GP; q++)
                        for (int tid = 0; tid < BA_NT; tid++) {
                            const uint16_t ow = S.GO[((sb * BA_KG + k) * BA_GP + q) * BA_NT + tid];
                            if (ow != 0xffffu) slots[ow].push_back((uint16_t)((k * BA_GP + q) * BA_NT + tid));
                        }
                size_t n = 0;
                for (int o = 0; o < S.nown; o++) {
                    S.csr_off[sb * (S.nown + 1) + o] = (uint16_t)n;
                    for (uint16_t sl : slots[o]) S.csr_idx[sb * BA_KG * BA_GP * BA_NT + n++] = sl;
                }
                S.csr_off[sb * (S.nown + 1) + S.nown] = (uint16_t)n;
            }
            // ---- riders: the pairs that are deep under a class, sorted by owner
            for (int cls = 0; cls < BA_NCLS; cls++) {
                std::vector<TTPair> dp;
                for (const TTPair &p : pairs) if (deep(cls, p)) dp.push_back(p);
                std::stable_sort(dp.begin(), dp.end(), [&](const TTPair &x, const TTPair &y) { return owner_of(x) < owner_of(y); });
                std::vector<uint4> &R = riders[(size_t)cls * 2 + b];
                uint16_t *cs = &S.r_csr[((size_t)cls * 2 + b) * (S.nown + 1)];
                size_t e = 0;
                for (int o = 0; o <= S.nown; o++) {
                    while (e < dp.size() && (int)owner_of(dp[e]) < o) e++;
                    cs[o] = (uint16_t)e;
                }
                for (const TTPair &p : dp) {
                    uint4 r;
                    r.x = bpack(cls, p);
                    r.y = Bof(tt_prepend((uint32_t)cls, BA_KB, p.cz), p.v) | (owner_of(p) << 16);
                    r.z = 8u * key_of(p);
                    r.w = 0u;
                    R.push_back(r);
                }
                rider_pairs[(size_t)cls * 2 + b] = dp;
            }
        }
        // ---- rider arrays, padded to a common capacity (multiple of 32)
        size_t mx = 0;
        for (auto &r : riders) mx = std::max(mx, r.size());
        S.nr = (int)((mx + 31) / 32 * 32);
        if (S.nr == 0) S.nr = 32;
        if (S.nr > BA_NT / 2) return;                          // two replicas of the rider set share the CTA
        S.R.assign((size_t)BA_NCLS * 2 * S.nr, make_uint4(0u, 0u, 0u, 0u));
        S.r_cnt.assign((size_t)BA_NCLS * 2, 0);
        S.R8.assign((size_t)BA_NCLS * 2 * 8 * S.nr, 0u);
        for (size_t i = 0; i < riders.size(); i++) {
            S.r_cnt[i] = (uint16_t)riders[i].size();
            std::copy(riders[i].begin(), riders[i].end(), S.R.begin() + i * S.nr);
            const int cls = (int)(i / 2);
            for (uint32_t hi = 0; hi < 8u; hi++)
                for (size_t e = 0; e < rider_pairs[i].size(); e++) {
                    const TTPair &p = rider_pairs[i][e];
                    const int lz = 31 - __builtin_clz(p.cz);
                    uint32_t x = 0;                            // B_8 = 0: |z| >= 1
                    for (int sft = 4; sft <= 7; sft++)
                        if (lz + sft <= m) x |= Bof(tt_prepend((hi << 4) | (uint32_t)cls, sft, p.cz), p.v) << (8 * (sft - 4));
                    S.R8[(i * 8 + hi) * S.nr + e] = x;
                }
        }
    }
    // ---- direct table of the pairs (v, empty): .x = 1 | B_1 << 8 | B_2 << 16 | B_3 << 24, .y = B_4 | .. | B_7 << 24 with
    // B_s = B(sigma_s, v) (B_0 = emb(empty, v) = 1; B_8 = [sigma_8 = v] is formed by the kernels) ---------------------
    T.EPS8.assign((size_t)256 * nv, make_uint2(0u, 0u));
    for (uint32_t sig = 0; sig < 256u; sig++)
        for (int v = 0; v < nv; v++) {
            uint32_t w[2] = {1u, 0u};
            for (int sft = 1; sft <= 7 && sft <= m; sft++)
                w[sft / 4] |= Bof((1u << sft) | (sig & ((1u << sft) - 1u)), v) << (8 * (sft % 4));
            T.EPS8[(size_t)sig * nv + v] = make_uint2(w[0], w[1]);
        }
    T.EPSH.assign((size_t)BA_NCLS * 8 * nv, 0u);
    for (uint32_t cls = 0; cls < BA_NCLS; cls++)
        for (uint32_t hi = 0; hi < 8u; hi++)
            for (int v = 0; v < nv; v++) T.EPSH[((size_t)cls * 8 + hi) * nv + v] = T.EPS8[(size_t)((hi << 4) | cls) * nv + v].y;
    T.ok = true;
}
