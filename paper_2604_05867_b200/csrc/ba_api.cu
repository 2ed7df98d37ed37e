// ba_api.cu -- C ABI of libba (include/ba.h): context, host-side tables, launch sequencing.
// Unity build: the kernels live in the .cuh files included below.
#include "../../include/ba.h"
#include "ba_internal.h"
#include "ba_tables.h"
#include "ba_enum_in.cuh"
#include "ba_enum_out.cuh"
#include "ba_stream.cuh"
#include "ba_fast.cuh"
#include "ba_peaks.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <memory>
#include <mutex>
#include <string>
#include <vector>

// ------------------------------------------------------------------------------------------------ ctx
struct ba_ctx {
    int n = 0, m = 0, h = 0, mode = BA_MODE_ENUM, sym = 0;
    double d = 0.0;
    size_t NX = 0, NY = 0, NZ = 0, napart = 0;
    KConst kc;
    cudaStream_t st = nullptr;
    bool own_buffers = false, own_stream = false;
    double *p = nullptr, *q = nullptr, *D = nullptr;
    unsigned char *scratch = nullptr;
    // carved from scratch
    double *c = nullptr, *crow = nullptr, *Hc = nullptr, *Apart = nullptr, *S = nullptr, *park = nullptr, *part = nullptr, *scal = nullptr, *hist = nullptr;
    GroupDev gin, gout;              // pair schedules of the two sweeps (device pointers into scratch)
    GroupDev ginf;                   // input sweep proper (IN_SWEEP): deep part of the chains in factored form, no riders
    uint2 *EPS8 = nullptr;
    uint32_t *LTV_off = nullptr, *LTV = nullptr;            // subsequences of every v (input sweep, pairs (v, empty))
    uint8_t *LT = nullptr;                                  // [2^m][2^{m+1}] emb(w, v) of the low tile (k_low_tile)
    uint32_t *EPSH = nullptr;
    double *elog = nullptr;
    unsigned int *counters = nullptr;
    unsigned long long *cnt = nullptr;
    size_t npart_cap = 0;
    bool hc_ready = false;
    long long iters = 0;
    int num_sms = 0, grid_in = 0, grid_out = 0, block = 0;
    size_t smem_in = 0, smem_out = 0;
    std::vector<cudaEvent_t> ev;     // 4 per timed iteration + 1
    cudaEvent_t ev_setup[2] = {nullptr, nullptr};      // around the one-off Hc pass
    int ev_iters = 0;
    std::string err;
};

static const char *g_static_err = "ba: invalid or null context";

static int fail(ba_ctx *c, int code, const std::string &msg) {
    if (c) c->err = msg;
    return code;
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(c, BA_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));          \
    } while (0)

static size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

// ------------------------------------------------------------------------------------------------ host helpers
static double host_binom(int n, int k) {
    double r = 1.0;
    for (int i = 1; i <= k; i++) r = r * (double)(n - k + i) / (double)i;
    return std::floor(r + 0.5);
}

// ------------------------------------------------------------------------------------------------ scratch layout
struct SideLayout { size_t GB, GA, GO, GW, csr_off, csr_idx, R, r_cnt, r_csr, R8; };
struct ScratchLayout {
    size_t c, crow, Hc, Apart, S, park, part, scal, hist, EPS8, EPSH, LT, LTV_off, LTV, elog, counters, cnt, total;
    SideLayout in, out, inf;
    size_t napart, npart_cap;
};

static int low_m(int n) { return n < BA_MLOW ? n : BA_MLOW; }

// The tile tables depend on m only and are immutable once built: one copy per process, built on first use.
static std::shared_ptr<const TileTables> tile_tables(int m) {
    static std::mutex mu;
    static std::shared_ptr<const TileTables> cache[BA_MLOW + 1];
    std::lock_guard<std::mutex> lk(mu);
    if (!cache[m]) {
        auto t = std::make_shared<TileTables>();
        build_tile_tables(m, *t);
        cache[m] = t;
    }
    return cache[m];
}

#define BA_MAX_GRID_IN 256             // CTAs of the input sweep that have a parking place for their accumulators
#define BA_FINAL_BLOCKS_PER_SM 8      // grid of k_in_final = SMs x this; one reduction triple per block

static void side_layout(const GroupSide &G, SideLayout &L, size_t &o) {
    L.GB = o; o += align256(G.GB.size() * 16);
    L.GA = o; o += align256(G.GA.size() * 4);
    L.GO = o; o += align256(G.GO.size() * 2);
    L.GW = o; o += align256(G.GW.size() * 2);
    L.csr_off = o; o += align256(G.csr_off.size() * 2);
    L.csr_idx = o; o += align256(G.csr_idx.size() * 2);
    L.R = o; o += align256(G.R.size() * 16);
    L.r_cnt = o; o += align256(G.r_cnt.size() * 2);
    L.r_csr = o; o += align256(G.r_csr.size() * 2);
    L.R8 = o; o += align256(G.R8.size() * 4);
}

static void scratch_layout(int n, const TileTables &T, ScratchLayout &L) {
    const int m = low_m(n), h = n - m;
    const size_t NX = (size_t)1 << n, NY = ((size_t)2 << n) - 1, NZ = ((size_t)2 << m) - 1;
    L.napart = (((size_t)2 << h) - 1) * NZ;
    size_t fastwords = 2 * (((size_t)2 << n) + 64);          // FAST mode ping-pong buffers
    if (L.napart < fastwords) L.napart = fastwords;
    L.npart_cap = 65536;                                     // >= grid of k_in_final
    size_t o = 0;
    L.c = o; o += align256((NY + 1) * 8);                    // c[code], entry 0 unused
    L.crow = o; o += align256(((size_t)4 << h) * ((size_t)1 << m) * 8);   // rows (code(y') <= 2^{h+1}-1, b) of 2^m operands
    L.Hc = o; o += align256(NX * 8);
    L.Apart = o; o += align256(L.napart * 8);
    L.S = o; o += align256(2 * NX * 8);                      // partial sums of the two lists (input sweep)
    L.park = o; o += align256((size_t)BA_MAX_GRID_IN * 2 * BA_NSLOT * BA_NT * 8);   // parked accumulators, one set per CTA of the input sweep
    L.part = o; o += align256(L.npart_cap * 3 * 8);
    L.scal = o; o += align256(8 * 8);
    L.hist = o; o += align256((size_t)BA_HIST_CAP * 3 * 8);
    L.EPS8 = o; o += align256(T.EPS8.size() * 8);
    L.EPSH = o; o += align256(T.EPSH.size() * 4);
    L.LT = o; o += align256(T.LT.size());
    L.LTV_off = o; o += align256(T.LTV_off.size() * 4);
    L.LTV = o; o += align256(T.LTV.size() * 4);
    L.elog = o; o += align256((size_t)BA_ELOG_N * 8);
    side_layout(T.in, L.in, o);
    side_layout(T.inf, L.inf, o);
    side_layout(T.out, L.out, o);
    L.counters = o; o += align256(16 * 4);
    L.cnt = o; o += align256(8 * 8);
    L.total = o;
}

extern "C" size_t ba_scratch_bytes(int n) {
    if (n < 1 || n > BA_NMAX) return 0;
    const std::shared_ptr<const TileTables> Tp = tile_tables(low_m(n));
    const TileTables &T = *Tp;
    if (!T.ok) return 0;
    ScratchLayout L;
    scratch_layout(n, T, L);
    return L.total;
}

extern "C" int ba_terms_per_sweep(int n, unsigned long long *T) {
    if (n < 1 || n > BA_NMAX || !T) return BA_EINVAL;
    unsigned long long tot = 0;
    for (int k = 0; k <= n; k++) {
        unsigned long long s = 0;
        for (int i = 0; i <= n - k; i++) s += (unsigned long long)host_binom(n, i);
        tot += s << k;
    }
    *T = tot;
    return BA_OK;
}

// Host-only self-check of the static tile tables of width m (include/ba.h): under every class, every pair
// (v, z != empty) of the m-bit deletion channel must be served exactly once, by a pair slot or by a rider, with
// the B_s an independent DP gives; the slots of a group must share their operand, and a warp's loop type must cover
// its slots.
static uint32_t chk_emb(uint32_t w, int lw, uint32_t v, int lv) {
    if (lw > lv) return 0;
    uint32_t e[BA_MLOW + 2];
    for (int r = 0; r <= lw; r++) e[r] = (r == 0);
    for (int i = 0; i < lv; i++)
        for (int r = lw; r >= 1; r--)
            if (((w >> (lw - r)) & 1u) == ((v >> (lv - 1 - i)) & 1u)) e[r] += e[r - 1];
    return e[lw];
}

extern "C" int ba_debug_check_tables(int m, unsigned long long stats[4]) {
    if (m < 1 || m > BA_MLOW || !stats) return BA_EINVAL;
    const std::shared_ptr<const TileTables> Tp = tile_tables(m);
    const TileTables &T = *Tp;
    if (!T.ok) return BA_EINVAL;
    const int nv = 1 << m, NZc = 2 << m;
    stats[0] = stats[1] = stats[2] = stats[3] = 0;
    auto Bs = [&](uint32_t sig, int s, uint32_t cz, int v) -> uint32_t {      // B(sigma_s.z, v)
        const int lz = 31 - __builtin_clz(cz);
        if (lz + s > m) return 0u;
        return chk_emb(((sig & ((1u << s) - 1u)) << lz) | (cz - (1u << lz)), lz + s, (uint32_t)v, m);
    };
    for (int side4 = 0; side4 < 3; side4++) {               // 0: input sweep tables, 1: output sweep tables; 2: the input
        const int side = side4 & 1;                         // sweep proper (IN_SWEEP), where the deep part of the chains is
        const bool fact = side4 >= 2;                       // summed in factored form, so there is no rider
        const GroupSide &G = (side4 == 0) ? T.in : (side4 == 1) ? T.out : T.inf;
        for (int cls = 0; cls < BA_NCLS; cls++)
            for (int b = 0; b < 2; b++) {
                std::vector<uint8_t> seen((size_t)nv * NZc, 0);
                // pos = operand position in the staged row (in: code(z[1:]), out: v); ow = owner (in: v, out: code(z))
                auto visit = [&](uint32_t pos, uint32_t ow, uint32_t b0123, int nb, const uint32_t *tail8) -> bool {
                    int v; uint32_t cz;
                    if (side) { v = (int)pos; cz = ow; }
                    else {
                        if (pos < 2 && (int)pos != b) return false;          // z = "b" sits at position b of the half row
                        const uint32_t tc = (pos < 2) ? 1u : pos;
                        const int lt = 31 - __builtin_clz(tc);
                        v = (int)ow; cz = (1u << (lt + 1)) | ((uint32_t)b << lt) | (tc - (1u << lt));
                    }
                    if (v < 0 || v >= nv || cz < 2 || cz >= (uint32_t)NZc) return false;
                    const int lz = 31 - __builtin_clz(cz);
                    if ((int)((cz >> (lz - 1)) & 1u) != b || seen[(size_t)v * NZc + cz]++) return false;
                    for (int s = 0; s < 4; s++) if (((b0123 >> (8 * s)) & 0xffu) != Bs((uint32_t)cls, s, cz, v)) return false;
                    if (nb == 4) return fact || Bs((uint32_t)cls, 4, cz, v) == 0;         // a slot pair must not be deep (enumerating tables)
                    for (uint32_t hi = 0; hi < 16u; hi++)                                 // rider: B_4 .. B_8
                        for (int s = 4; s <= 8; s++) {
                            const uint32_t want = Bs((hi << 4) | (uint32_t)cls, s, cz, v);
                            const uint32_t got = (s == 8) ? 0u : ((tail8[hi] >> (8 * (s - 4))) & 0xffu);
                            if (want != got || (s == 4 && got != (uint32_t)nb - 5u)) return false;
                        }
                    return true;
                };
                for (int k = 0; k < BA_KG; k++)
                    for (int tid = 0; tid < BA_NT; tid++) {
                        const uint4 e4 = G.GB[(((size_t)cls * 2 + b) * BA_KG + k) * BA_NT + tid];
                        const uint32_t e[4] = {e4.x, e4.y, e4.z, e4.w};
                        const size_t sb = (size_t)((G.nsc == BA_NCLS) ? cls : (G.nsc == 2) ? (cls & 1) : 0) * 2 + b;
                        const uint32_t pos = G.GA[(sb * BA_KG + k) * BA_NT + tid] >> 3;
                        const int hm = (G.GW[sb * (BA_NT / 32) + tid / 32] >> (8 * (k / 2))) & 0xff;    // the half of group k
                        for (int q = 0; q < BA_GP; q++) {
                            const uint32_t ow = G.GO[((sb * BA_KG + k) * BA_GP + q) * BA_NT + tid];
                            if (!(e[q] & 0xffu)) { if (e[q]) return BA_EINVAL; continue; }      // unused, or deep under this class
                            if (ow == 0xffffu || (k & 1) >= (hm & 3)) return BA_EINVAL;         // the half's loop must reach the slot
                            if ((hm >> 2) == 2 && (e[q] >> 16)) return BA_EINVAL;               // a type-2 loop ignores B_2, B_3
                            if ((hm >> 2) == 1 && (e[q] >> 8)) return BA_EINVAL;                // a type-1 loop ignores B_1..B_3
                            if (!visit(pos, ow, e[q], 4, nullptr)) return BA_EINVAL;
                            if (!fact) stats[side ? 2 : 0]++;
                        }
                    }
                const int nr = G.r_cnt[cls * 2 + b];
                if (fact && nr != 0) return BA_EINVAL;
                for (int e = 0; e < nr; e++) {
                    const uint4 rd = G.R[((size_t)cls * 2 + b) * G.nr + e];
                    uint32_t tail8[16];
                    for (uint32_t hi = 0; hi < 16u; hi++) tail8[hi] = G.R8[(((size_t)cls * 2 + b) * 8 + (hi & 7u)) * G.nr + e];   // B_4..B_7 read sigma bits 4..6 only
                    if (!visit(rd.z >> 3, rd.y >> 16, rd.x, 5 + (int)(rd.y & 0xffu), tail8) || (rd.y & 0xffu) == 0) return BA_EINVAL;
                    const uint16_t *cs = &G.r_csr[((size_t)cls * 2 + b) * (G.nown + 1)];
                    const uint32_t ow = rd.y >> 16;
                    if (!(cs[ow] <= e && e < cs[ow + 1])) return BA_EINVAL;                     // the epilogue finds it under its owner
                    stats[side ? 3 : 1]++;
                }
                for (int v = 0; v < nv; v++)                 // nothing missing
                    for (uint32_t cz = 2; cz < (uint32_t)NZc; cz++) {
                        const int lz = 31 - __builtin_clz(cz);
                        if ((int)((cz >> (lz - 1)) & 1u) != b) continue;
                        if ((chk_emb(cz - (1u << lz), lz, (uint32_t)v, m) != 0) != (seen[(size_t)v * NZc + cz] != 0)) return BA_EINVAL;
                    }
            }
        // the epilogue's CSR lists every used slot exactly once, under its owner (per schedule and list)
        for (int sb = 0; sb < G.nsc * 2; sb++) {
            std::vector<uint8_t> hit((size_t)BA_NSLOT * BA_NT, 0);
            for (int o = 0; o < G.nown; o++)
                for (int q = G.csr_off[(size_t)sb * (G.nown + 1) + o]; q < G.csr_off[(size_t)sb * (G.nown + 1) + o + 1]; q++) {
                    const uint32_t sl = G.csr_idx[(size_t)sb * BA_NSLOT * BA_NT + q];
                    const int kq = (int)(sl / BA_NT), tid = (int)(sl % BA_NT);
                    if (G.GO[(((size_t)sb * BA_KG + kq / BA_GP) * BA_GP + kq % BA_GP) * BA_NT + tid] != o || hit[sl]++) return BA_EINVAL;
                }
            for (int k = 0; k < BA_KG; k++)
                for (int q = 0; q < BA_GP; q++)
                    for (int tid = 0; tid < BA_NT; tid++)
                        if ((G.GO[(((size_t)sb * BA_KG + k) * BA_GP + q) * BA_NT + tid] != 0xffffu) != (hit[(size_t)(k * BA_GP + q) * BA_NT + tid] != 0)) return BA_EINVAL;
        }
    }
    return BA_OK;
}

// ------------------------------------------------------------------------------------------------ create / destroy
static int setup_ctx(ba_ctx *c, int n, double d) {
    c->n = n; c->m = low_m(n); c->h = n - c->m; c->d = d;
    c->NX = (size_t)1 << n; c->NY = ((size_t)2 << n) - 1; c->NZ = ((size_t)2 << c->m) - 1;
    KConst &kc = c->kc;
    kc.n = n; kc.m = c->m; kc.h = c->h; kc.klen = -1;
    for (int k = 0; k <= BA_NMAX_I; k++) { kc.w[k] = 0.0; kc.lebar[k] = 0.0; }
    for (int k = 0; k <= n; k++) {
        long double a = 1.0L, b = 1.0L;                      // 0^0 = 1 (R7)
        for (int i = 0; i < k; i++) a *= (long double)(1.0 - d);
        for (int i = 0; i < n - k; i++) b *= (long double)d;
        kc.w[k] = (double)(a * b);
        kc.lebar[k] = std::log2(host_binom(n, k)) - (double)k;
    }
    return BA_OK;
}

template <typename V>
static cudaError_t upload(void *dst, const std::vector<V> &src, cudaStream_t st) {
    if (src.empty()) return cudaSuccess;
    return cudaMemcpyAsync(dst, src.data(), src.size() * sizeof(V), cudaMemcpyHostToDevice, st);
}

static cudaError_t upload_side(unsigned char *s, const GroupSide &G, const SideLayout &L, GroupDev &D, cudaStream_t st) {
    cudaError_t e;
    if ((e = upload(s + L.GB, G.GB, st)) != cudaSuccess) return e;
    if ((e = upload(s + L.GA, G.GA, st)) != cudaSuccess) return e;
    if ((e = upload(s + L.GO, G.GO, st)) != cudaSuccess) return e;
    if ((e = upload(s + L.GW, G.GW, st)) != cudaSuccess) return e;
    if ((e = upload(s + L.csr_off, G.csr_off, st)) != cudaSuccess) return e;
    if ((e = upload(s + L.csr_idx, G.csr_idx, st)) != cudaSuccess) return e;
    if ((e = upload(s + L.R, G.R, st)) != cudaSuccess) return e;
    if ((e = upload(s + L.r_cnt, G.r_cnt, st)) != cudaSuccess) return e;
    if ((e = upload(s + L.r_csr, G.r_csr, st)) != cudaSuccess) return e;
    if ((e = upload(s + L.R8, G.R8, st)) != cudaSuccess) return e;
    D.GB = (const uint4 *)(s + L.GB); D.GA = (const uint32_t *)(s + L.GA); D.GO = (const uint16_t *)(s + L.GO);
    D.GW = (const uint16_t *)(s + L.GW); D.csr_off = (const uint16_t *)(s + L.csr_off); D.csr_idx = (const uint16_t *)(s + L.csr_idx);
    D.R = (const uint4 *)(s + L.R); D.r_cnt = (const uint16_t *)(s + L.r_cnt); D.r_csr = (const uint16_t *)(s + L.r_csr);
    D.R8 = (const uint32_t *)(s + L.R8);
    D.nr = G.nr; D.nown = G.nown; D.nsc = G.nsc;
    return cudaSuccess;
}

// MaxDynamicSharedMemorySize is per-function state shared by every ctx of the process: only ever raise it, so that
// one ctx cannot shrink what another live ctx launches with.
static cudaError_t raise_smem_limits(size_t smem_in, size_t smem_out) {
    static std::mutex mu;
    static size_t max_in = 0, max_out = 0;
    std::lock_guard<std::mutex> lk(mu);
    if (smem_in > max_in) max_in = smem_in;
    if (smem_out > max_out) max_out = smem_out;
    cudaError_t e;
#define BA_SET(k, v) if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(v))) != cudaSuccess) return e
    BA_SET(k_enum_in<IN_SWEEP>, max_in); BA_SET(k_enum_in<IN_HC>, max_in); BA_SET(k_enum_in<IN_DEBUG>, max_in); BA_SET(k_enum_in<IN_COUNT>, max_in);
    BA_SET(k_enum_out<OUT_SWEEP>, max_out); BA_SET(k_enum_out<OUT_DEBUG>, max_out); BA_SET(k_enum_out<OUT_COUNT>, max_out);
#undef BA_SET
    return cudaSuccess;
}

static int finish_create(ba_ctx *c) {
    const std::shared_ptr<const TileTables> Tp = tile_tables(c->m);
    const TileTables &T = *Tp;
    if (!T.ok) return fail(c, BA_EINVAL, "internal: tile tables do not fit their packed formats");
    ScratchLayout L;
    scratch_layout(c->n, T, L);
    unsigned char *s = c->scratch;
    c->c = (double *)(s + L.c); c->crow = (double *)(s + L.crow); c->Hc = (double *)(s + L.Hc); c->Apart = (double *)(s + L.Apart); c->S = (double *)(s + L.S); c->park = (double *)(s + L.park);
    c->part = (double *)(s + L.part); c->scal = (double *)(s + L.scal); c->hist = (double *)(s + L.hist);
    c->EPS8 = (uint2 *)(s + L.EPS8); c->EPSH = (uint32_t *)(s + L.EPSH); c->elog = (double *)(s + L.elog); c->LT = (uint8_t *)(s + L.LT);
    c->LTV_off = (uint32_t *)(s + L.LTV_off); c->LTV = (uint32_t *)(s + L.LTV);
    c->counters = (unsigned int *)(s + L.counters); c->cnt = (unsigned long long *)(s + L.cnt);
    c->napart = L.napart; c->npart_cap = L.npart_cap;

    CK(upload(c->EPS8, T.EPS8, c->st));
    CK(upload(c->LT, T.LT, c->st));
    CK(upload(c->LTV_off, T.LTV_off, c->st));
    CK(upload(c->LTV, T.LTV, c->st));
    CK(upload(c->EPSH, T.EPSH, c->st));
    std::vector<double> elog(BA_ELOG_N, 0.0);
    for (int e = 2; e < BA_ELOG_N; e++) elog[e] = (double)((long double)e * log2l((long double)e));
    CK(upload(c->elog, elog, c->st));
    CK(upload_side(s, T.in, L.in, c->gin, c->st));
    CK(upload_side(s, T.inf, L.inf, c->ginf, c->st));
    CK(upload_side(s, T.out, L.out, c->gout, c->st));
    CK(cudaMemsetAsync(c->c, 0, 8, c->st));                  // c[0] is never written by k_out_final
    uint32_t hb[BA_NMAX_I + 1][BA_NMAX_I + 1];
    for (int a = 0; a <= BA_NMAX_I; a++)
        for (int b = 0; b <= BA_NMAX_I; b++) hb[a][b] = (b <= a) ? (uint32_t)host_binom(a, b) : 0u;
    CK(cudaMemcpyToSymbolAsync(c_binom, hb, sizeof(hb), 0, cudaMemcpyHostToDevice, c->st));
    CK(cudaStreamSynchronize(c->st));                        // T and hb go out of scope

    int dev = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev));
    c->block = BA_NT;
    c->smem_in = std::max(enum_in_smem(c->gin.nr, false).total, enum_in_smem(c->ginf.nr, true).total);
    c->smem_out = enum_out_smem(c->gout.nr).total;
    CK(raise_smem_limits(c->smem_in, c->smem_out));
    int occ_in = 1, occ_out = 1;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_in, k_enum_in<IN_SWEEP>, c->block, c->smem_in));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_out, k_enum_out<OUT_SWEEP>, c->block, c->smem_out));
    if (occ_in < 1 || occ_out < 1) return fail(c, BA_ECUDA, "ENUM kernels do not fit on an SM");
    size_t items_in = (size_t)2 << c->h, items_out = 2 * (((size_t)2 << c->h) - 1);      // (high part, list) pairs
    size_t gi = (size_t)c->num_sms * occ_in, go = (size_t)c->num_sms * occ_out;
    c->grid_in = (int)(items_in < gi ? items_in : gi);
    if (c->grid_in > BA_MAX_GRID_IN) c->grid_in = BA_MAX_GRID_IN;
    c->grid_out = (int)(items_out < go ? items_out : go);

    // p0 uniform
    k_fill<<<c->num_sms * 4, 256, 0, c->st>>>(c->NX, c->p, 1.0 / (double)c->NX);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(c->st));
    return BA_OK;
}

extern "C" int ba_create_ext(int n, double d, void *p_dev, void *q_dev, void *D_dev, void *scratch_dev,
                             size_t scratch_bytes, void *cuda_stream, ba_ctx **out) {
    if (out) *out = nullptr;
    if (!out || n < 1 || n > BA_NMAX || !(d >= 0.0 && d <= 1.0) || !p_dev || !q_dev || !D_dev || !scratch_dev)
        return BA_EINVAL;
    if (scratch_bytes < ba_scratch_bytes(n) || ((uintptr_t)scratch_dev & 255u)) return BA_ENOMEM;
    ba_ctx *c = new (std::nothrow) ba_ctx();
    if (!c) return BA_ENOMEM;
    setup_ctx(c, n, d);
    c->p = (double *)p_dev; c->q = (double *)q_dev; c->D = (double *)D_dev;
    c->scratch = (unsigned char *)scratch_dev;
    c->st = (cudaStream_t)cuda_stream;
    int rc = finish_create(c);
    if (rc) { delete c; return rc; }
    *out = c;
    return BA_OK;
}

extern "C" int ba_create(int n, double d, ba_ctx **out) {
    if (out) *out = nullptr;
    if (!out || n < 1 || n > BA_NMAX || !(d >= 0.0 && d <= 1.0)) return BA_EINVAL;
    ba_ctx *c = new (std::nothrow) ba_ctx();
    if (!c) return BA_ENOMEM;
    setup_ctx(c, n, d);
    c->own_buffers = true;
    size_t sb = ba_scratch_bytes(n);
    int rc = BA_OK;
    if (cudaMalloc(&c->p, c->NX * 8) != cudaSuccess || cudaMalloc(&c->q, c->NY * 8) != cudaSuccess ||
        cudaMalloc(&c->D, c->NX * 8) != cudaSuccess || cudaMalloc(&c->scratch, sb) != cudaSuccess)
        rc = BA_ENOMEM;
    if (!rc && cudaStreamCreateWithFlags(&c->st, cudaStreamNonBlocking) != cudaSuccess) rc = BA_ECUDA;
    else c->own_stream = (rc == BA_OK);
    if (!rc) rc = finish_create(c);
    if (rc) { cudaGetLastError(); ba_destroy(c); return rc; }
    *out = c;
    return BA_OK;
}

extern "C" void ba_destroy(ba_ctx *c) {
    if (!c) return;
    if (c->st || !c->own_stream) cudaStreamSynchronize(c->st);
    for (auto e : c->ev) cudaEventDestroy(e);
    for (auto e : c->ev_setup) if (e) cudaEventDestroy(e);
    if (c->own_buffers) { cudaFree(c->p); cudaFree(c->q); cudaFree(c->D); cudaFree(c->scratch); }
    if (c->own_stream && c->st) cudaStreamDestroy(c->st);
    delete c;
}

extern "C" const char *ba_last_error(const ba_ctx *c) { return c ? c->err.c_str() : g_static_err; }

static bool host_symmetric(const double *p, size_t NX) {
    for (size_t x = 0; x < NX / 2; x++)
        if (p[x] != p[NX - 1 - x]) return false;
    return true;
}

extern "C" int ba_set_symmetry(ba_ctx *c, int on) {
    if (!c) return BA_EINVAL;
    if (on != 0 && on != 1) return fail(c, BA_EINVAL, "ba_set_symmetry: on must be 0 or 1");
    if (on && c->h < 1) return fail(c, BA_EINVAL, "ba_set_symmetry: needs n >= 9 (a high part of at least one bit)");
    if (on && c->mode != BA_MODE_ENUM) return fail(c, BA_EINVAL, "ba_set_symmetry: only in BA_MODE_ENUM (FAST iterations do not keep p(x) == p(~x) bit for bit)");
    if (on) {                                               // the current p must be complement-symmetric, bit for bit
        std::vector<double> hp(c->NX);
        CK(cudaMemcpyAsync(hp.data(), c->p, c->NX * 8, cudaMemcpyDeviceToHost, c->st));
        CK(cudaStreamSynchronize(c->st));
        if (!host_symmetric(hp.data(), c->NX)) return fail(c, BA_EINVAL, "ba_set_symmetry: p(x) != p(~x) for some x");
    }
    c->sym = on;
    return BA_OK;
}

extern "C" int ba_set_exact(ba_ctx *c, int k) {
    if (!c) return BA_EINVAL;
    if (k < 0 || k > c->n) return fail(c, BA_EINVAL, "ba_set_exact: k outside [0, n]");
    if (c->iters != 0) return fail(c, BA_ESTATE, "ba_set_exact: only before the first iteration");
    for (int j = 0; j <= c->n; j++) c->kc.w[j] = 0.0;
    c->kc.w[k] = 1.0 / host_binom(c->n, k);                 // P_{n,k}(y|x) = emb(y,x) / C(n,k)
    c->kc.klen = k;                                         // the sweeps skip the nodes / prefixes that cannot reach length k
    c->hc_ready = false;                                    // Hc depends on the weights
    return BA_OK;
}

extern "C" int ba_set_mode(ba_ctx *c, int mode) {
    if (!c) return BA_EINVAL;
    if (mode != BA_MODE_ENUM && mode != BA_MODE_FAST) return fail(c, BA_EINVAL, "ba_set_mode: unknown mode");
    if (mode == BA_MODE_FAST && c->sym) return fail(c, BA_EINVAL, "ba_set_mode: BA_MODE_FAST is refused while complement symmetry is on (ba_set_symmetry(c, 0) first)");
    c->mode = mode;
    return BA_OK;
}

// ------------------------------------------------------------------------------------------------ launches
static InArgs make_in_args(ba_ctx *c) {
    InArgs a;
    a.kc = c->kc; a.g = c->gin; a.EPS8 = c->EPS8; a.EPSH = c->EPSH; a.LTV_off = c->LTV_off; a.LTV = c->LTV;
    a.c = c->c; a.crow = c->crow; a.elog = c->elog; a.S = c->S; a.park = c->park;
    a.counter = c->counters; a.sym = 0; a.dbg_x = 0; a.dbg_out = nullptr; a.cnt = c->cnt;
    return a;
}

static OutArgs make_out_args(ba_ctx *c) {
    OutArgs a;
    a.kc = c->kc; a.g = c->gout; a.EPS8 = c->EPS8;
    a.p = c->p; a.M = c->S; a.Apart = c->Apart; a.counter = c->counters + 4; a.sym = 0; a.dbg_item = 0; a.dbg_cz = 0; a.dbg_out = nullptr;
    a.cnt = c->cnt + 2;
    return a;
}

// Hc(x) = sum_y w_k emb(y,x) log2(emb(y,x)/ebar_k): one enumerating pass, independent of the iterate.
static int ensure_hc(ba_ctx *c) {
    if (c->hc_ready) return BA_OK;
    for (int i = 0; i < 2; i++) if (!c->ev_setup[i]) CK(cudaEventCreate(&c->ev_setup[i]));
    CK(cudaEventRecord(c->ev_setup[0], c->st));
    CK(cudaMemsetAsync(c->counters, 0, 16 * 4, c->st));
    InArgs a = make_in_args(c);
    // Hc does not depend on the iterate and the channel is invariant under complementing x and y together (Theorem 4,
    // P:785-791, g = cpl): Hc(~x) = Hc(x) whatever p is.  So the pass always enumerates only the inputs whose leading
    // symbol is 0 (whenever there is a high part) and k_hc_final mirrors them.
    const int hsym = (c->h >= 1) ? 1 : 0;
    a.sym = hsym;
    k_enum_in<IN_HC><<<c->grid_in, c->block, c->smem_in, c->st>>>(a);
    CK(cudaGetLastError());
    const long double K = 0.0L;                             // the pass centres term by term
    k_hc_final<<<c->num_sms * 8, 256, 0, c->st>>>(c->NX, c->S, c->S + c->NX, c->Hc, hsym, (double)K);
    CK(cudaGetLastError());
    CK(cudaEventRecord(c->ev_setup[1], c->st));
    c->hc_ready = true;
    return BA_OK;
}

static int launch_out_sweep(ba_ctx *c) {
    if (c->mode == BA_MODE_ENUM) {
        CK(cudaMemsetAsync(c->counters + 4, 0, 4, c->st));
        OutArgs a = make_out_args(c);
        a.sym = c->sym;
        // M(u, w) of the low tile, for the pairs (v, empty) of the sweep.  It lives in S: the partial sums of the input
        // sweep are dead from k_in_final to the next input sweep, and 2^h * 2^{m+1} = 2 * 2^n entries is their size.
        const size_t NU = (size_t)1 << c->h;
        const size_t ltb = (NU + BA_LT_UB - 1) / BA_LT_UB;
        k_low_tile<<<(unsigned)(ltb < (size_t)c->num_sms * 16 ? ltb : (size_t)c->num_sms * 16), 512, 0, c->st>>>(c->m, NU, c->p, c->LT, c->S);
        CK(cudaGetLastError());
        k_enum_out<OUT_SWEEP><<<c->grid_out, c->block, c->smem_out, c->st>>>(a);
        CK(cudaGetLastError());
        k_out_final<<<c->num_sms * 8, 256, 0, c->st>>>(c->kc, c->Apart, nullptr, c->q, c->c, c->crow, c->sym);
        CK(cudaGetLastError());
    } else {
        double *buf0 = c->Apart, *buf1 = c->Apart + (((size_t)2 << c->n) + 64);
        const double *in = c->p;
        double *out = buf0;
        for (int s = 0; s < c->n; s++) {
            k_fast_fwd<<<c->num_sms * 8, 256, 0, c->st>>>(c->n, s, in, out);
            CK(cudaGetLastError());
            in = out;
            out = (out == buf0) ? buf1 : buf0;
        }
        k_out_final<<<c->num_sms * 8, 256, 0, c->st>>>(c->kc, nullptr, in, c->q, c->c, c->crow, 0);
        CK(cudaGetLastError());
    }
    return BA_OK;
}

static int launch_in_sweep(ba_ctx *c, size_t *npart) {
    int nb = c->num_sms * BA_FINAL_BLOCKS_PER_SM;
    if ((size_t)nb > c->NX / 256 + 1) nb = (int)(c->NX / 256 + 1);
    if (c->mode == BA_MODE_ENUM) {
        CK(cudaMemsetAsync(c->counters, 0, 4, c->st));
        InArgs a = make_in_args(c);
        a.g = c->ginf;                                      // the sweep's own schedule: no riders, deep part factored
        a.sym = c->sym;
        k_enum_in<IN_SWEEP><<<c->grid_in, c->block, c->smem_in, c->st>>>(a);
        CK(cudaGetLastError());
        k_in_final<<<nb, 256, 0, c->st>>>(c->NX, c->Hc, c->S, c->S + c->NX, c->p, c->D, c->part, c->sym);
        CK(cudaGetLastError());
    } else {
        double *buf0 = c->Apart, *buf1 = c->Apart + (((size_t)2 << c->n) + 64);
        const double *in = c->c + 1;                          // c is stored by code: idx(y) = code(y) - 1
        double *out = buf0;
        for (int s = c->n - 1; s >= 0; s--) {
            k_fast_bwd<<<c->num_sms * 8, 256, 0, c->st>>>(c->n, s, in, out);
            CK(cudaGetLastError());
            in = out;
            out = (out == buf0) ? buf1 : buf0;
        }
        k_in_final<<<nb, 256, 0, c->st>>>(c->NX, c->Hc, in, nullptr, c->p, c->D, c->part, 0);
        CK(cudaGetLastError());
    }
    *npart = (size_t)nb;
    return BA_OK;
}

extern "C" int ba_iterate(ba_ctx *c, int k) {
    if (!c) return BA_EINVAL;
    if (k < 0) return fail(c, BA_EINVAL, "ba_iterate: k < 0");
    if (k == 0) return BA_OK;
    int rc = ensure_hc(c);
    if (rc) return rc;
    const int timed = k < 64 ? k : 64;                 // time the last `timed` iterations
    while ((int)c->ev.size() < 4 * timed + 1) {
        cudaEvent_t e;
        CK(cudaEventCreate(&e));
        c->ev.push_back(e);
    }
    c->ev_iters = timed;
    for (int it = 0; it < k; it++) {
        const int ti = it - (k - timed);
        if (ti >= 0) CK(cudaEventRecord(c->ev[4 * ti], c->st));
        rc = launch_out_sweep(c);
        if (rc) return rc;
        if (ti >= 0) CK(cudaEventRecord(c->ev[4 * ti + 1], c->st));
        size_t npart = 0;
        rc = launch_in_sweep(c, &npart);
        if (rc) return rc;
        if (ti >= 0) CK(cudaEventRecord(c->ev[4 * ti + 2], c->st));
        const int slot = (int)(c->iters % BA_HIST_CAP);
        k_finalize<<<1, 1024, 0, c->st>>>(c->part, npart, c->scal, c->hist, slot);
        CK(cudaGetLastError());
        k_update<<<c->num_sms * 8, 256, 0, c->st>>>(c->NX, c->p, c->D, c->scal);
        CK(cudaGetLastError());
        if (ti >= 0) CK(cudaEventRecord(c->ev[4 * ti + 3], c->st));
        c->iters++;
    }
    CK(cudaEventRecord(c->ev[4 * timed], c->st));
    return BA_OK;
}

extern "C" int ba_last_timing(ba_ctx *c, double ms[4]) {
    if (!c || !ms) return BA_EINVAL;
    if (c->ev_iters <= 0) return fail(c, BA_ESTATE, "ba_last_timing: no iteration yet");
    CK(cudaStreamSynchronize(c->st));
    double acc[4] = {0, 0, 0, 0};
    for (int t = 0; t < c->ev_iters; t++) {
        float f;
        CK(cudaEventElapsedTime(&f, c->ev[4 * t], c->ev[4 * t + 1])); acc[0] += f;
        CK(cudaEventElapsedTime(&f, c->ev[4 * t + 1], c->ev[4 * t + 2])); acc[1] += f;
        CK(cudaEventElapsedTime(&f, c->ev[4 * t + 2], c->ev[4 * t + 3])); acc[2] += f;
    }
    float tot;
    CK(cudaEventElapsedTime(&tot, c->ev[0], c->ev[4 * c->ev_iters]));
    for (int i = 0; i < 3; i++) ms[i] = acc[i] / c->ev_iters;
    ms[3] = tot / c->ev_iters;
    return BA_OK;
}

// ------------------------------------------------------------------------------------------------ getters / setters
extern "C" int ba_bounds(ba_ctx *c, double *I_lower, double *maxD_upper) {
    if (!c || !I_lower || !maxD_upper) return c ? fail(c, BA_EINVAL, "ba_bounds: null pointer") : BA_EINVAL;
    if (c->iters == 0) return fail(c, BA_ESTATE, "ba_bounds: no iteration yet");
    double h3[3];
    const int slot = (int)((c->iters - 1) % BA_HIST_CAP);
    CK(cudaMemcpyAsync(h3, c->hist + 3 * slot, 24, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    *I_lower = h3[0];
    *maxD_upper = h3[1];
    if (!std::isfinite(h3[0]) || !std::isfinite(h3[1]))
        return fail(c, BA_ENUMERIC, "ba_bounds: non-finite bound (q(y)=0 or p underflow, see DESIGN.md G8)");
    return BA_OK;
}

extern "C" int ba_stats(ba_ctx *c, double *log2Z, long long *iters_done) {
    if (!c) return BA_EINVAL;
    if (iters_done) *iters_done = c->iters;
    if (log2Z) {
        if (c->iters == 0) return fail(c, BA_ESTATE, "ba_stats: no iteration yet");
        const int slot = (int)((c->iters - 1) % BA_HIST_CAP);
        CK(cudaMemcpyAsync(log2Z, c->hist + 3 * slot + 2, 8, cudaMemcpyDeviceToHost, c->st));
        CK(cudaStreamSynchronize(c->st));
    }
    return BA_OK;
}

extern "C" int ba_get_history(ba_ctx *c, int count, double *out) {
    if (!c || !out || count < 0) return c ? fail(c, BA_EINVAL, "ba_get_history: bad argument") : BA_EINVAL;
    if ((long long)count > c->iters || count > BA_HIST_CAP) return fail(c, BA_EINVAL, "ba_get_history: count too large");
    if (count > 0) {                                        // the ring wraps at most once: one or two contiguous copies
        const int first = (int)((c->iters - count) % BA_HIST_CAP);
        const int n1 = (first + count <= BA_HIST_CAP) ? count : BA_HIST_CAP - first;
        CK(cudaMemcpyAsync(out, c->hist + 3 * (size_t)first, (size_t)n1 * 24, cudaMemcpyDeviceToHost, c->st));
        if (n1 < count) CK(cudaMemcpyAsync(out + 3 * (size_t)n1, c->hist, (size_t)(count - n1) * 24, cudaMemcpyDeviceToHost, c->st));
    }
    CK(cudaStreamSynchronize(c->st));
    return BA_OK;
}

extern "C" int ba_get_p(ba_ctx *c, double *p_host) {
    if (!c || !p_host) return c ? fail(c, BA_EINVAL, "ba_get_p: null pointer") : BA_EINVAL;
    CK(cudaMemcpyAsync(p_host, c->p, c->NX * 8, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    return BA_OK;
}

extern "C" int ba_get_q(ba_ctx *c, double *q_host) {
    if (!c || !q_host) return c ? fail(c, BA_EINVAL, "ba_get_q: null pointer") : BA_EINVAL;
    if (c->iters == 0) return fail(c, BA_ESTATE, "ba_get_q: no iteration yet");
    CK(cudaMemcpyAsync(q_host, c->q, c->NY * 8, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    return BA_OK;
}

extern "C" int ba_get_D(ba_ctx *c, double *D_host) {
    if (!c || !D_host) return c ? fail(c, BA_EINVAL, "ba_get_D: null pointer") : BA_EINVAL;
    if (c->iters == 0) return fail(c, BA_ESTATE, "ba_get_D: no iteration yet");
    CK(cudaMemcpyAsync(D_host, c->D, c->NX * 8, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    return BA_OK;
}

extern "C" int ba_set_p(ba_ctx *c, const double *p_host) {
    if (!c || !p_host) return c ? fail(c, BA_EINVAL, "ba_set_p: null pointer") : BA_EINVAL;
    long double sum = 0.0L;
    for (size_t i = 0; i < c->NX; i++) {
        const double v = p_host[i];
        if (!std::isfinite(v) || !(v > 0.0)) return fail(c, BA_EINVAL, "ba_set_p: entry not finite and positive");
        sum += v;
    }
    if (fabsl(sum - 1.0L) > 1e-9L) return fail(c, BA_EINVAL, "ba_set_p: |sum p - 1| > 1e-9");
    if (c->sym && !host_symmetric(p_host, c->NX))
        return fail(c, BA_EINVAL, "ba_set_p: complement symmetry is on (ba_set_symmetry) and p(x) != p(~x) for some x");
    CK(cudaMemcpyAsync(c->p, p_host, c->NX * 8, cudaMemcpyHostToDevice, c->st));
    CK(cudaStreamSynchronize(c->st));
    return BA_OK;
}

// ------------------------------------------------------------------------------------------------ debug
extern "C" int ba_debug_emb_row(ba_ctx *c, unsigned x, unsigned *emb_out) {
    if (!c || !emb_out) return c ? fail(c, BA_EINVAL, "ba_debug_emb_row: null pointer") : BA_EINVAL;
    if ((size_t)x >= c->NX) return fail(c, BA_EINVAL, "ba_debug_emb_row: x out of range");
    uint32_t *dev = nullptr;
    CK(cudaMalloc(&dev, c->NY * 4));
    cudaError_t e = cudaMemsetAsync(dev, 0, c->NY * 4, c->st);
    if (e == cudaSuccess) {
        InArgs a = make_in_args(c);
        a.dbg_x = x; a.dbg_out = dev;
        k_enum_in<IN_DEBUG><<<2, c->block, c->smem_in, c->st>>>(a);      // one CTA per list
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(emb_out, dev, c->NY * 4, cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    cudaFree(dev);
    if (e != cudaSuccess) return fail(c, BA_ECUDA, std::string("ba_debug_emb_row: ") + cudaGetErrorString(e));
    return BA_OK;
}

extern "C" int ba_debug_emb_col(ba_ctx *c, unsigned yidx, unsigned *emb_out) {
    if (!c || !emb_out) return c ? fail(c, BA_EINVAL, "ba_debug_emb_col: null pointer") : BA_EINVAL;
    if ((size_t)yidx >= c->NY) return fail(c, BA_EINVAL, "ba_debug_emb_col: yidx out of range");
    uint32_t *dev = nullptr;
    CK(cudaMalloc(&dev, c->NX * 4));
    cudaError_t e = cudaMemsetAsync(dev, 0, c->NX * 4, c->st);
    const uint32_t cyt = yidx + 1u;                          // code of the target y
    const int ky = 31 - __builtin_clz(cyt);
    for (int j = 0; j <= c->m && j <= ky && e == cudaSuccess; j++) {   // the splits y = y'.z, |z| = j
        if (ky - j > c->h) continue;
        OutArgs a = make_out_args(c);
        a.dbg_item = cyt >> j;
        a.dbg_cz = (1u << j) | (cyt & ((1u << j) - 1u));
        a.dbg_out = dev;
        k_enum_out<OUT_DEBUG><<<1, c->block, c->smem_out, c->st>>>(a);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(emb_out, dev, c->NX * 4, cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    cudaFree(dev);
    if (e != cudaSuccess) return fail(c, BA_ECUDA, std::string("ba_debug_emb_col: ") + cudaGetErrorString(e));
    return BA_OK;
}

extern "C" int ba_debug_count_terms(ba_ctx *c, unsigned long long *in_terms, unsigned long long *out_terms,
                                    unsigned long long *in_emb_sum, unsigned long long *out_emb_sum) {
    if (!c) return BA_EINVAL;
    CK(cudaMemsetAsync(c->counters, 0, 16 * 4, c->st));
    CK(cudaMemsetAsync(c->cnt, 0, 8 * 8, c->st));
    InArgs ia = make_in_args(c);
    k_enum_in<IN_COUNT><<<c->grid_in, c->block, c->smem_in, c->st>>>(ia);
    CK(cudaGetLastError());
    OutArgs oa = make_out_args(c);
    k_enum_out<OUT_COUNT><<<c->grid_out, c->block, c->smem_out, c->st>>>(oa);
    CK(cudaGetLastError());
    unsigned long long h4[4];
    CK(cudaMemcpyAsync(h4, c->cnt, 32, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    if (in_terms) *in_terms = h4[0];
    if (in_emb_sum) *in_emb_sum = h4[1];
    if (out_terms) *out_terms = h4[2];
    if (out_emb_sum) *out_emb_sum = h4[3];
    return BA_OK;
}

// ------------------------------------------------------------------------------------------------ measured peaks
template <int KIND>
static cudaError_t run_peak(int sms, int iters, unsigned long long *clk_dev, double *sink_dev, double *per_clk_sm, double *mhz) {
    k_peak<KIND><<<sms, 512>>>(clk_dev, sink_dev, 16, 12345u);                 // warm-up (instruction cache, clocks)
    cudaEvent_t e0, e1;
    cudaError_t e;
    if ((e = cudaEventCreate(&e0)) != cudaSuccess) return e;
    if ((e = cudaEventCreate(&e1)) != cudaSuccess) { cudaEventDestroy(e0); return e; }
    cudaEventRecord(e0);
    k_peak<KIND><<<sms, 512>>>(clk_dev, sink_dev, iters, 12345u);
    cudaEventRecord(e1);
    e = cudaDeviceSynchronize();
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess) return e;
    std::vector<unsigned long long> h(sms);
    if ((e = cudaMemcpy(h.data(), clk_dev, (size_t)sms * 8, cudaMemcpyDeviceToHost)) != cudaSuccess) return e;
    double avg = 0;
    for (auto v : h) avg += (double)v;
    avg /= sms;
    *per_clk_sm = (double)iters * 32.0 * 16.0 / avg;                            // 32 instructions per iteration, 16 warps
    *mhz = avg / (ms * 1e-3) / 1e6;
    return cudaSuccess;
}

extern "C" int ba_measure_peaks(double out[6]) {
    if (!out) return BA_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1)
        return BA_ECUDA;
    unsigned long long *clk = nullptr;
    double *sink = nullptr;
    if (cudaMalloc(&clk, (size_t)sms * 8) != cudaSuccess) return BA_ENOMEM;
    if (cudaMalloc(&sink, 8) != cudaSuccess) { cudaFree(clk); return BA_ENOMEM; }
    double mhz[4] = {0, 0, 0, 0};
    cudaError_t e = run_peak<PK_DFMA>(sms, 4000, clk, sink, &out[0], &mhz[0]);
    if (e == cudaSuccess) e = run_peak<PK_IDP>(sms, 4000, clk, sink, &out[1], &mhz[1]);
    if (e == cudaSuccess) e = run_peak<PK_LDS64>(sms, 4000, clk, sink, &out[2], &mhz[2]);
    if (e == cudaSuccess) e = run_peak<PK_FFMA>(sms, 8000, clk, sink, &out[3], &mhz[3]);
    cudaFree(clk); cudaFree(sink);
    if (e != cudaSuccess) { cudaGetLastError(); return BA_ECUDA; }
    out[4] = (mhz[0] + mhz[1] + mhz[2] + mhz[3]) / 4.0;
    out[5] = (double)sms;
    return BA_OK;
}

extern "C" int ba_setup_ms(ba_ctx *c, double *ms_host) {
    if (!c || !ms_host) return c ? fail(c, BA_EINVAL, "ba_setup_ms: null pointer") : BA_EINVAL;
    if (!c->hc_ready) return fail(c, BA_ESTATE, "ba_setup_ms: no iteration yet");
    CK(cudaStreamSynchronize(c->st));
    float f = 0.f;
    CK(cudaEventElapsedTime(&f, c->ev_setup[0], c->ev_setup[1]));
    *ms_host = (double)f;
    return BA_OK;
}

// ------------------------------------------------------------------------------------------------ no-allocation entry point
// ba_in_final_noalloc (ba.h): the epilogue of the input sweep -- D = Hc - (S0 + S1) and the reductions of 8(a3),
// for callers that must not allocate (CUDA graph capture, serving loops).  k_in_final keeps its
// first-stage partials in ctx-owned scratch (`part`, cudaMalloc'ed by ba_create); this variant keeps them in the
// file-scope device array below: 48 KB that every GPU which loads the library holds until exit.  Its name is a
// host-side stand-in in host code, so the device address is taken once per device with cudaGetSymbolAddress
// and handed to the kernels.
#define BA_NA_CHUNK ((size_t)1 << 15)                          // inputs per block: fixed, so the sums have one order per n
static __device__ __align__(256) double g_na_part[3 * BA_NOALLOC_MAXBLK];

__global__ void __launch_bounds__(256) k_in_final_na(size_t NX, const double *__restrict__ Hc, const double *__restrict__ S0,
                                                     const double *__restrict__ S1, const double *__restrict__ p,
                                                     double *__restrict__ D, double *__restrict__ part) {
    __shared__ double sr[3 * 8];
    double r0 = 0.0, r1 = -INFINITY, r2 = 0.0;
    const size_t lo = (size_t)blockIdx.x * BA_NA_CHUNK, hi = (lo + BA_NA_CHUNK < NX) ? lo + BA_NA_CHUNK : NX;
    for (size_t i = lo + threadIdx.x; i < hi; i += blockDim.x) {
        const double Dx = Hc[i] - (S1 ? S0[i] + S1[i] : S0[i]);
        D[i] = Dx;
        const double px = p[i];
        r0 += px * Dx; r1 = fmax(r1, Dx); r2 += px * exp2(Dx);
    }
    for (int o = 16; o > 0; o >>= 1) {
        r0 += __shfl_xor_sync(0xffffffffu, r0, o);
        r1 = fmax(r1, __shfl_xor_sync(0xffffffffu, r1, o));
        r2 += __shfl_xor_sync(0xffffffffu, r2, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sr[warp * 3] = r0; sr[warp * 3 + 1] = r1; sr[warp * 3 + 2] = r2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t0 = 0.0, t1 = -INFINITY, t2 = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) { t0 += sr[w * 3]; t1 = fmax(t1, sr[w * 3 + 1]); t2 += sr[w * 3 + 2]; }
        part[(size_t)blockIdx.x * 3] = t0; part[(size_t)blockIdx.x * 3 + 1] = t1; part[(size_t)blockIdx.x * 3 + 2] = t2;
    }
}

// second stage: the npart triples of the scratch, in a fixed order, to out3 = {sum p D, max D, sum p 2^D}
__global__ void __launch_bounds__(1024) k_finalize_na(const double *__restrict__ part, int npart, double *__restrict__ out3) {
    __shared__ double s0[1024], s1[1024], s2[1024];
    const int tid = threadIdx.x;
    double a0 = 0.0, a1 = -INFINITY, a2 = 0.0;
    for (int i = tid; i < npart; i += 1024) { a0 += part[3 * i]; a1 = fmax(a1, part[3 * i + 1]); a2 += part[3 * i + 2]; }
    s0[tid] = a0; s1[tid] = a1; s2[tid] = a2;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if (tid < o) { s0[tid] += s0[tid + o]; s1[tid] = fmax(s1[tid], s1[tid + o]); s2[tid] += s2[tid + o]; }
        __syncthreads();
    }
    if (tid == 0) { out3[0] = s0[0]; out3[1] = s1[0]; out3[2] = s2[0]; }
}

#define BA_NA_MAXDEV 64
static std::mutex g_na_mu;
static double *g_na_ptr[BA_NA_MAXDEV];                         // device address of g_na_part, per device (null = not taken yet)
static thread_local char g_na_err[256] = "";

static int na_fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_na_err, sizeof g_na_err, fmt, ap);
    va_end(ap);
    return code;
}

extern "C" const char *ba_noalloc_last_error(void) { return g_na_err; }

extern "C" int ba_in_final_noalloc(int n, const void *Hc_dev, const void *S0_dev, const void *S1_dev, const void *p_dev,
                                   void *D_dev, void *out3_dev, void *stream) {
    if (n < 1 || n > BA_NOALLOC_NMAX)
        return na_fail(BA_EINVAL, "ba_in_final_noalloc: n = %d is outside [1, %d]: the static scratch holds %d block partials of %zu inputs each",
                       n, BA_NOALLOC_NMAX, BA_NOALLOC_MAXBLK, BA_NA_CHUNK);
    if (!Hc_dev || !S0_dev || !p_dev || !D_dev || !out3_dev) return na_fail(BA_EINVAL, "ba_in_final_noalloc: null pointer");
    const size_t NX = (size_t)1 << n;
    const int nblk = (int)((NX + BA_NA_CHUNK - 1) / BA_NA_CHUNK);
    if (nblk > BA_NOALLOC_MAXBLK) return na_fail(BA_EINVAL, "ba_in_final_noalloc: %d blocks exceed the static scratch (%d)", nblk, BA_NOALLOC_MAXBLK);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(BA_ECUDA, "ba_in_final_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= BA_NA_MAXDEV) return na_fail(BA_EINVAL, "ba_in_final_noalloc: device ordinal %d not below %d", dev, BA_NA_MAXDEV);
    double *part = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_na_mu);
        if (!g_na_ptr[dev]) {                                  // once per device, with that device current
            void *sym = nullptr;
            e = cudaGetSymbolAddress(&sym, g_na_part);
            if (e != cudaSuccess || !sym) {
                cudaGetLastError();
                return na_fail(BA_ECUDA, "ba_in_final_noalloc: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
            }
            g_na_ptr[dev] = (double *)sym;
        }
        part = g_na_ptr[dev];
    }
    cudaStream_t st = (cudaStream_t)stream;
    // every triple the second stage reads is written by the first stage of the same call: nothing has to start at zero
    k_in_final_na<<<nblk, 256, 0, st>>>(NX, (const double *)Hc_dev, (const double *)S0_dev, (const double *)S1_dev,
                                        (const double *)p_dev, (double *)D_dev, part);
    k_finalize_na<<<1, 1024, 0, st>>>(part, nblk, (double *)out3_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(BA_ECUDA, "ba_in_final_noalloc: launch: %s", cudaGetErrorString(e));
    g_na_err[0] = 0;
    return BA_OK;
}
