// ba_tables.h -- host-side construction of the static low tables and pair schedules of the ENUM
// kernels (formats: ba_internal.h).  Everything here depends on m = min(n, 8) only.
#pragma once
#include "ba_internal.h"

#include <algorithm>
#include <vector>

struct TileTables {
    int m = 0, nv = 0;
    std::vector<uint2> T64;            // v-major pairs {W, P}; entries [0, BA_C) are the all-zero dummy chunk
    std::vector<uint32_t> vbase;       // [nv] entry index of v's list (its null entry)
    std::vector<uint2> in_desc;        // [2][BA_NC][BA_NT]
    std::vector<uint16_t> in_csr_off;  // [nv + 1]
    std::vector<uint16_t> in_csr_idx;  // accumulator slots (b*BA_NC + slot)*BA_NT + thread of v's chunks
    std::vector<uint2> Tz;             // z-major pairs {W, P'}; entries [0, BA_C) all-zero
    std::vector<uint32_t> Wv;          // W words of T64 (chain walks of the output sweep)
    std::vector<uint2> out_desc;       // [2][BA_NC][BA_NT]
    std::vector<uint16_t> out_csr_off; // [2^{m+1}] indexed by code(z) - 1 (entry 0, the empty z, has no chunks)
    std::vector<uint16_t> out_csr_idx;
    bool ok = false;
};

static inline uint32_t tt_emb(uint32_t z, int lz, uint32_t v, int lv) {   // #embeddings of z in v (textbook DP)
    uint32_t e[BA_MLOW + 2];
    for (int r = 0; r <= lz; r++) e[r] = (r == 0);
    for (int i = 0; i < lv; i++) {
        const uint32_t vb = (v >> (lv - 1 - i)) & 1u;
        for (int r = lz; r >= 1; r--)
            if (((z >> (lz - r)) & 1u) == vb) e[r] += e[r - 1];
    }
    return e[lz];
}

struct TTChunk { int key, owner, first; };   // key = chain bound m - min|z|; owner = v or code(z); first = entry index

static inline void tt_assign(std::vector<TTChunk> &ch, int b, uint32_t stride, bool in_side, const std::vector<uint32_t> &vbase,
                             std::vector<uint2> &desc, std::vector<std::vector<uint16_t>> &owner_slots) {
    std::stable_sort(ch.begin(), ch.end(), [](const TTChunk &x, const TTChunk &y) {
        return x.key != y.key ? x.key < y.key : x.owner < y.owner;
    });
    for (size_t k = 0; k < ch.size(); k++) {
        const int slot = (int)(k / BA_NT), thr = (int)(k % BA_NT);
        const size_t di = ((size_t)b * BA_NC + slot) * BA_NT + thr;
        uint2 d;
        d.x = (uint32_t)ch[k].first * stride | ((uint32_t)ch[k].owner << 20) | 0x80000000u;
        d.y = in_side ? vbase[ch[k].owner] * stride : 0u;
        desc[di] = d;
        owner_slots[ch[k].owner].push_back((uint16_t)di);
    }
}

static inline void build_tile_tables(int m, TileTables &T) {
    const int nv = 1 << m;
    T.m = m; T.nv = nv; T.ok = false;
    // ---- v-major lists ------------------------------------------------------------------------
    struct Ent { uint32_t code; uint32_t B; };
    std::vector<std::vector<Ent>> lst(nv);                 // local index -> entry (code 0 = null / padding)
    std::vector<std::vector<int>> loc(nv);                 // code(z) -> local index, 0 if absent
    std::vector<int> start[2];
    start[0].assign(nv, 0); start[1].assign(nv, 0);
    std::vector<int> cnt[2];
    cnt[0].assign(nv, 0); cnt[1].assign(nv, 0);
    T.vbase.assign(nv, 0);
    uint32_t total = BA_C;                                 // dummy chunk first
    for (int v = 0; v < nv; v++) {
        std::vector<Ent> &L = lst[v];
        L.push_back({0u, 0u});                             // null
        L.push_back({1u, 1u});                             // empty string, B = 1
        for (int b = 0; b < 2; b++) {
            start[b][v] = (int)L.size();
            for (int lz = m; lz >= 1; lz--)                // longest first: short chains first
                for (uint32_t z = 0; z < (1u << lz); z++) {
                    if ((int)((z >> (lz - 1)) & 1u) != b) continue;
                    const uint32_t B = tt_emb(z, lz, (uint32_t)v, m);
                    if (B) { L.push_back({(1u << lz) | z, B}); cnt[b][v]++; }
                }
            while ((L.size() - start[b][v]) % BA_C) L.push_back({0u, 0u});
        }
        if (L.size() > 255) return;                        // local links are 8 bit
        loc[v].assign((size_t)2 << m, 0);
        for (size_t i = 1; i < L.size(); i++)
            if (L[i].code) loc[v][L[i].code] = (int)i;
        T.vbase[v] = total;
        total += (uint32_t)L.size();
    }
    if ((size_t)total * 8 >= (1u << 20) || (size_t)total * 4 >= (1u << 16)) return;
    T.T64.assign(total, make_uint2(0u, 0u));
    T.Wv.assign(total, 0u);
    for (int v = 0; v < nv; v++)
        for (size_t i = 1; i < lst[v].size(); i++) {
            const uint32_t cz = lst[v][i].code;
            if (!cz) continue;
            const int lz = 31 - __builtin_clz(cz);
            const uint32_t zval = cz - (1u << lz);
            uint32_t W = 0;
            if (lz + 1 <= m)
                for (uint32_t b = 0; b < 2; b++) {
                    const uint32_t cbz = (1u << (lz + 1)) | (b << lz) | zval;
                    const int li = loc[v][cbz];
                    if (li) W |= ((uint32_t)li | (lst[v][li].B << 8)) << (16 * b);
                }
            const uint32_t P = lst[v][i].B | ((uint32_t)lz << 8) | ((8u * cz) << 16);
            T.T64[T.vbase[v] + i] = make_uint2(W, P);
            T.Wv[T.vbase[v] + i] = W;
        }
    // ---- input-sweep schedule: chunks of BA_C consecutive pairs of one v -------------------------
    T.in_desc.assign((size_t)2 * BA_NC * BA_NT, make_uint2(0u, 0u));
    std::vector<std::vector<uint16_t>> vslots(nv);
    for (int b = 0; b < 2; b++) {
        std::vector<TTChunk> ch;
        for (int v = 0; v < nv; v++)
            for (int i = 0; i * BA_C < cnt[b][v]; i++) {
                const int first = start[b][v] + i * BA_C;
                int last = std::min(cnt[b][v], (i + 1) * BA_C) - 1;
                const uint32_t czl = lst[v][start[b][v] + last].code;
                ch.push_back({m - (31 - __builtin_clz(czl)), v, (int)T.vbase[v] + first});
            }
        if (ch.size() > (size_t)BA_NC * BA_NT) return;
        tt_assign(ch, b, 8u, true, T.vbase, T.in_desc, vslots);
    }
    T.in_csr_off.assign(nv + 1, 0);
    T.in_csr_idx.clear();
    for (int v = 0; v < nv; v++) {
        T.in_csr_off[v] = (uint16_t)T.in_csr_idx.size();
        for (uint16_t s : vslots[v]) T.in_csr_idx.push_back(s);
    }
    T.in_csr_off[nv] = (uint16_t)T.in_csr_idx.size();
    // ---- z-major table and output-sweep schedule ------------------------------------------------
    const int NZc = 2 << m;                                // codes 1 .. 2^{m+1}-1
    T.Tz.assign(BA_C, make_uint2(0u, 0u));
    T.out_desc.assign((size_t)2 * BA_NC * BA_NT, make_uint2(0u, 0u));
    std::vector<std::vector<uint16_t>> zslots(NZc);
    for (int b = 0; b < 2; b++) {
        std::vector<TTChunk> ch;
        for (int lz = m; lz >= 1; lz--)
            for (uint32_t z = 0; z < (1u << lz); z++) {
                if ((int)((z >> (lz - 1)) & 1u) != b) continue;
                const uint32_t cz = (1u << lz) | z;
                const int first = (int)T.Tz.size();
                int nsup = 0;
                for (int v = 0; v < nv; v++) {
                    const int li = loc[v][cz];
                    if (!li) continue;
                    const uint32_t Pp = lst[v][li].B | ((uint32_t)v << 8) | ((4u * T.vbase[v]) << 16);
                    T.Tz.push_back(make_uint2(T.Wv[T.vbase[v] + li], Pp));
                    nsup++;
                }
                while ((T.Tz.size() - first) % BA_C) T.Tz.push_back(make_uint2(0u, 0u));
                for (int i = 0; i * BA_C < nsup; i++) ch.push_back({m - lz, (int)cz, first + i * BA_C});
            }
        if (ch.size() > (size_t)BA_NC * BA_NT) return;
        tt_assign(ch, b, 8u, false, T.vbase, T.out_desc, zslots);
    }
    if (T.Tz.size() * 8 >= (1u << 20)) return;
    T.out_csr_off.assign(NZc, 0);
    T.out_csr_idx.clear();
    for (int cz = 1; cz < NZc; cz++) {
        T.out_csr_off[cz - 1] = (uint16_t)T.out_csr_idx.size();
        for (uint16_t s : zslots[cz]) T.out_csr_idx.push_back(s);
    }
    T.out_csr_off[NZc - 1] = (uint16_t)T.out_csr_idx.size();
    T.ok = true;
}
