/*
 * ba_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU Blahut-Arimoto (BA) for the finite-length
 * binary deletion channel BDC_d^n, written from the paper (PAPER.md, "P:line")
 * and BASELINE.json:north_star.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may use it.  It shares no
 * code, header, table or constant with the CUDA path.
 *
 *   channel law   W(y|x) = emb(y,x) (1-d)^{|y|} d^{n-|y|}          (north_star)
 *   emb(y,x)      "#times y appears as a subsequence of x"
 *                 counted here by brute force over all 2^n keep-masks (north_star).
 *   BA step 1     q(y) = sum_x p(x) W(y|x)
 *   BA step 2(a)  log W^(t)(x) = sum_y W(y|x) log( p(x) W(y|x) / q(y) )   (log form P:189-193)
 *                 => D(x) = sum_y W(y|x) log2( W(y|x)/q(y) ) = log2 W^(t)(x) - log2 p(x)
 *   BA step 2(b)  p'(x) = p(x) 2^{D(x)} / Z,  Z = sum_x p(x) 2^{D(x)}
 *   bounds        I(p) = sum_x p(x) D(x)  <=  C_n(d)  <=  max_x D(x)      (north_star)
 *   log base 2 everywhere.
 *
 * Readings:
 *   R2  x in [0,2^n); the bit at paper position i (0 = leftmost) is (x>>(n-1-i))&1.
 *       idx(y) = (2^{|y|}-1) + val(y), val = y read MSB-first; idx(empty)=0.
 *   R3  the empty string is an output; emb(empty,x)=1.
 *   R5  entries with emb=0 contribute nothing (0 log 0 = 0).
 *   R7  0^0 = 1 for w_k at d=0 or d=1; lengths with w_k=0 carry no mass.
 *   R9  every sum uses a long double accumulator in ascending index order; q, D, p are
 *       rounded to double and stored, so each iteration starts from FP64 state.
 *   G8  update is p' = max(p 2^D / Z, 2^-1000) (never active in the parity configs).
 *
 * Parity pins: tests/test_oracle_pins.py (closed forms, invariants, brute force) --
 * every function below is pinned there, the G8 floor line of orc_ba_step included
 * (test_floor_G8_*); nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_EINVAL -1
#define ORC_ENOMEM -2

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_weights(int n, double d, double *w);

/* O2: dense output index of the string with `len` bits and MSB-first value `val` (R2, a5). */
static inline uint64_t orc_idx(int len, uint64_t val) { return (((uint64_t)1 << len) - 1) + val; }

/* length of the output with dense index j: largest k with 2^k - 1 <= j */
static inline int orc_len_of_idx(uint64_t j) {
    int k = 0;
    while ((((uint64_t)1 << (k + 1)) - 1) <= j) k++;
    return k;
}

/*
 * O3: E[x*NY + idx(y)] = emb(y,x) by brute force over keep-masks (north_star).
 * For every mask m in [0,2^n): y = the bits of x at the set positions of m, in order.
 * E must hold 2^n * (2^{n+1}-1) uint32, caller-allocated.
 */
int orc_emb_dense(int n, uint32_t *E) {
    if (n < 1 || n > 15 || !E) return ORC_EINVAL;
    const uint64_t NX = (uint64_t)1 << n, NY = ((uint64_t)1 << (n + 1)) - 1;
    memset(E, 0, NX * NY * sizeof(uint32_t));
#pragma omp parallel for schedule(static)
    for (int64_t x = 0; x < (int64_t)NX; x++) {
        uint32_t *row = E + (uint64_t)x * NY;
        for (uint64_t m = 0; m < NX; m++) {
            uint64_t val = 0;
            int len = 0;
            for (int i = 0; i < n; i++) {            /* paper position i, left to right */
                int sh = n - 1 - i;
                if ((m >> sh) & 1) {
                    val = (val << 1) | (((uint64_t)x >> sh) & 1);
                    len++;
                }
            }
            row[orc_idx(len, val)] += 1;
        }
    }
    return ORC_OK;
}

/*
 * O3 for ONE input x, at sizes the dense matrix cannot reach (n <= 30): row[idx(y)] = emb(y,x), by the
 * same keep-mask enumeration as orc_emb_dense ("#times y appears as a subsequence of x").
 * row must hold 2^{n+1}-1 uint32, caller-allocated; it is zero-filled here.  Cost n 2^n.
 */
int orc_emb_row(int n, uint32_t x, uint32_t *row) {
    if (n < 1 || n > 30 || !row || ((uint64_t)x >> n) != 0) return ORC_EINVAL;
    const uint64_t NX = (uint64_t)1 << n, NY = ((uint64_t)1 << (n + 1)) - 1;
    memset(row, 0, NY * sizeof(uint32_t));
    for (uint64_t m = 0; m < NX; m++) {
        uint64_t val = 0;
        int len = 0;
        for (int i = 0; i < n; i++) {                /* paper position i, left to right */
            int sh = n - 1 - i;
            if ((m >> sh) & 1) {
                val = (val << 1) | (((uint64_t)x >> sh) & 1);
                len++;
            }
        }
        row[orc_idx(len, val)] += 1;
    }
    return ORC_OK;
}

/*
 * Divergence of ONE input from its emb row and an output distribution q (P:189-193 minus log2 p(x); R5):
 *   D(x) = sum_{j: row[j]>0} W_j (log2 W_j - log2 q(j)),  W_j = row[j] w_{len(j)},  w_k = (1-d)^k d^{n-k}.
 * The plain definition, one term per non-zero entry, long double accumulator, ascending j (R9).
 * Entries whose weight w_k is 0 are skipped (R7).  *nterms = number of non-zero emb entries.
 */
int orc_D_row(int n, double d, const uint32_t *row, const double *q, double *D_out, int64_t *nterms) {
    if (n < 1 || n > 30 || !row || !q || !D_out) return ORC_EINVAL;
    double w[64];
    int rc = orc_weights(n, d, w);
    if (rc) return rc;
    const uint64_t NY = ((uint64_t)1 << (n + 1)) - 1;
    long double acc = 0.0L;
    int64_t cnt = 0;
    for (uint64_t j = 0; j < NY; j++) {
        if (!row[j]) continue;
        cnt++;
        double wv = (double)row[j] * w[orc_len_of_idx(j)];
        if (wv != 0.0) acc += (long double)wv * (log2l((long double)wv) - log2l((long double)q[j]));
    }
    *D_out = (double)acc;
    if (nterms) *nterms = cnt;
    return ORC_OK;
}

/* O4: w_k = (1-d)^k d^{n-k}, with 0^0 = 1 (R7). w has n+1 entries. */
int orc_weights(int n, double d, double *w) {
    if (n < 1 || !(d >= 0.0 && d <= 1.0) || !w) return ORC_EINVAL;
    for (int k = 0; k <= n; k++) {
        long double a = 1.0L, b = 1.0L;
        for (int i = 0; i < k; i++) a *= (long double)(1.0 - d);
        for (int i = 0; i < n - k; i++) b *= (long double)d;
        w[k] = (double)(a * b);
    }
    return ORC_OK;
}

/* O4: explicit channel matrix W[x*NY + j] = E[x*NY + j] * w_{len(j)} (north_star). */
int orc_channel_from_emb(int n, double d, const uint32_t *E, double *W) {
    if (n < 1 || n > 15 || !E || !W) return ORC_EINVAL;
    double w[64];
    int rc = orc_weights(n, d, w);
    if (rc) return rc;
    const uint64_t NX = (uint64_t)1 << n, NY = ((uint64_t)1 << (n + 1)) - 1;
#pragma omp parallel for schedule(static)
    for (int64_t x = 0; x < (int64_t)NX; x++)
        for (uint64_t j = 0; j < NY; j++)
            W[(uint64_t)x * NY + j] = (double)E[(uint64_t)x * NY + j] * w[orc_len_of_idx(j)];
    return ORC_OK;
}

/*
 * O5: one BA iteration over an explicit NX x NY channel matrix W (row-major, rows = inputs).
 *   q(j)  = sum_x p(x) W[x][j]
 *   D(x)  = sum_{j: W[x][j]>0} W[x][j] (log2 W[x][j] - log2 q(j))   (P:189-193 minus log2 p(x); R5)
 *   I = sum_x p(x) D(x);  U = max_x D(x);  Z = sum_x p(x) 2^{D(x)}   (north_star)
 *   p'(x) = max(p(x) 2^{D(x)} / Z, 2^-1000)                         (G8)
 * stats = {I, U, log2 Z}.  q (NY), D (NX), p_next (NX) are outputs; p_next may alias p.
 * Long double accumulators, ascending index order, results rounded to double (R9).
 */
int orc_ba_step(int64_t NX, int64_t NY, const double *W, const double *p,
                double *q, double *D, double *stats, double *p_next) {
    if (NX < 1 || NY < 1 || !W || !p || !q || !D || !stats || !p_next) return ORC_EINVAL;
    long double *lq = (long double *)malloc((size_t)NY * sizeof(long double));
    if (!lq) return ORC_ENOMEM;

    /* step 1: output distribution; every thread owns a range of outputs j, x ascending */
#pragma omp parallel
    {
#ifdef _OPENMP
        int nt = omp_get_num_threads(), id = omp_get_thread_num();
#else
        int nt = 1, id = 0;
#endif
        int64_t j0 = NY * id / nt, j1 = NY * (id + 1) / nt;
        long double *acc = (long double *)calloc((size_t)(j1 - j0 + 1), sizeof(long double));
        for (int64_t x = 0; x < NX; x++) {
            const double *row = W + x * NY;
            long double px = (long double)p[x];
            for (int64_t j = j0; j < j1; j++)
                if (row[j] != 0.0) acc[j - j0] += px * (long double)row[j];
        }
        for (int64_t j = j0; j < j1; j++) {
            q[j] = (double)acc[j - j0];
            lq[j] = (q[j] > 0.0) ? log2l((long double)q[j]) : -INFINITY;
        }
        free(acc);
    }

    /* step 2(a): divergence per input */
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t x = 0; x < NX; x++) {
        const double *row = W + x * NY;
        long double acc = 0.0L;
        for (int64_t j = 0; j < NY; j++) {
            double wv = row[j];
            if (wv != 0.0) acc += (long double)wv * (log2l((long double)wv) - lq[j]);
        }
        D[x] = (double)acc;
    }
    free(lq);

    /* bounds and normaliser, serial, ascending x */
    long double I = 0.0L, Z = 0.0L;
    double U = -INFINITY;
    for (int64_t x = 0; x < NX; x++) {
        I += (long double)p[x] * (long double)D[x];
        Z += (long double)p[x] * exp2l((long double)D[x]);
        if (D[x] > U) U = D[x];
    }
    stats[0] = (double)I;
    stats[1] = U;
    stats[2] = (double)log2l(Z);

    /* step 2(b): normalised update with the G8 floor */
    const long double floor_p = ldexpl(1.0L, -1000);
    for (int64_t x = 0; x < NX; x++) {
        long double v = (long double)p[x] * exp2l((long double)D[x]) / Z;
        if (v < floor_p) v = floor_p;
        p_next[x] = (double)v;
    }
    return ORC_OK;
}

/*
 * O1/O6: K iterations from p0.  hist (3*K doubles) receives {I_t, U_t, log2 Z_t} for t=0..K-1.
 * On return p = p_K, q = q_{K-1}, D = D_{K-1} (R6).
 */
int orc_ba_run(int64_t NX, int64_t NY, const double *W, const double *p0, int K,
               double *hist, double *p, double *q, double *D) {
    if (K < 0 || !p0 || !p) return ORC_EINVAL;
    if (p != p0) memcpy(p, p0, (size_t)NX * sizeof(double));
    for (int t = 0; t < K; t++) {
        double st[3];
        int rc = orc_ba_step(NX, NY, W, p, q, D, st, p);
        if (rc) return rc;
        if (hist) { hist[3 * t] = st[0]; hist[3 * t + 1] = st[1]; hist[3 * t + 2] = st[2]; }
    }
    return ORC_OK;
}
