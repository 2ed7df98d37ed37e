/*
 * ba.h -- C ABI of libba: Blahut-Arimoto (BA) for the finite-length binary deletion channel
 * BDC_d^n on one NVIDIA B200 (sm_100a).  Hand-written CUDA kernels behind plain pointers;
 * no torch types, no exceptions, no mutable global state (see "Device"), no CPU fallback.
 *
 * Citations: "P:line" = PAPER.md line (arxiv 2604.05867); "NS" = BASELINE.json:north_star;
 * "R#/G#" = readings listed in DESIGN.md.
 *
 * Channel (NS): inputs x in {0,1}^n, outputs y in {0,1}^{<=n},
 *     W(y|x) = emb(y,x) (1-d)^{|y|} d^{n-|y|},  emb = #embeddings of y in x as a subsequence.
 * One BA iteration t (log form P:189-193), all logs base 2:
 *     q_t(y) = sum_x p_t(x) W(y|x)                      output sweep  (gather over supersequences, NS)
 *     D_t(x) = sum_y W(y|x) log2( W(y|x) / q_t(y) )     input sweep   (distinct subsequences of x, NS)
 *     I_t = sum_x p_t(x) D_t(x),  U_t = max_x D_t(x),  Z_t = sum_x p_t(x) 2^{D_t(x)}
 *     p_{t+1}(x) = max( p_t(x) 2^{D_t(x)} / Z_t , 2^-1000 )            (floor: G8)
 *     I_t <= C_n(d) <= U_t   (NS);  C(d) <= C_n(d)/n   (Lemma 1)
 *
 * Layout (R2): x is an integer in [0,2^n) whose bit (n-1-i) is the paper's x_i
 * (position 0 = leftmost = most significant).  Output y of length k and MSB-first value v has the
 * dense index idx(y) = (2^k - 1) + v; idx(empty) = 0; q has 2^{n+1}-1 entries.  All probability
 * arrays are FP64.
 *
 * Which iterate (R6): after a total of K >= 1 iterations, ba_bounds/ba_stats return
 * (I_{K-1}, U_{K-1}, log2 Z_{K-1}), ba_get_q / ba_get_D return q_{K-1}, D_{K-1}, ba_get_p returns p_K.
 *
 * Device: a ctx lives on the CUDA device that was current when it was created; the caller keeps that device current
 * (cudaSetDevice) for every call on the ctx.  The library keeps no global state besides an immutable, lazily built
 * cache of the static pair tables and the per-kernel shared-memory limit, which is only ever raised.
 *
 * Errors: every function returns BA_OK (0) or a negative code; nothing is printed, thrown or aborted.
 * ba_last_error(ctx) gives a ctx-owned message for the last failure on that ctx (static string if ctx
 * is NULL).  A ctx is not thread-safe; distinct ctxs are independent.
 *
 * Ownership: ba_create allocates device memory that ba_destroy frees.  ba_create_ext borrows the
 * caller's device buffers and CUDA stream, which must outlive the ctx.  Host buffers are caller-owned
 * and caller-sized.  Pointers documented "host" must be host-accessible, "device" device-accessible.
 */
#ifndef BA_H
#define BA_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ba_ctx ba_ctx;

enum {
    BA_OK = 0,
    BA_EINVAL = -1,   /* bad n, d, k, index, null pointer, non-normalised / non-positive p          */
    BA_ENOMEM = -2,   /* host or device allocation failed, or caller scratch too small               */
    BA_ECUDA = -3,    /* CUDA runtime error; text in ba_last_error                                    */
    BA_ESTATE = -4,   /* bounds / q / D requested before any iteration                                */
    BA_ENUMERIC = -5  /* non-finite bound (some q(y) = 0 or p underflow, G8)                          */
};

enum {
    BA_MODE_ENUM = 0, /* contract path (NS): the supersequences of every y / the distinct subsequences of every x are
                         enumerated once per sweep with their integer embedding counts.  A term (x,y), x = u.v, y = y'.z,
                         has emb = sum_s alpha_s B(sigma_s.z, v) (P:181 at the boundary of the low 8 positions): the
                         sweeps form s <= 3 term by term; the pairs with z empty (3.9 % of the terms) and, in the input
                         sweep, the tail s >= 4 are summed in factored form with the same identity.
                         The debug entry points below still produce every emb, bit for bit. */
    BA_MODE_FAST = 1  /* position-by-position deletion transform, O(n 2^n)/sweep  */
};

#define BA_NMAX 30    /* uint32 string codes; run to n = 28 in ENUM mode (profiles/) */

/* ---- required by the north star -------------------------------------------------------------- */

/* New problem (n in [1,BA_NMAX], d in [0,1]); p_0 uniform.  Library-owned device buffers and
 * stream.  *out is NULL on failure. */
int ba_create(int n, double d, ba_ctx **out);

/* Enqueue k >= 0 full BA iterations (both sweeps, reductions, update) on the ctx stream.  Does not
 * synchronise with the host. */
int ba_iterate(ba_ctx *c, int k);

/* Bounds in bits for C_n(d) from the last completed iteration (R6): I_lower = I(p) (NS),
 * maxD_upper = max_x D(x).  Synchronises the stream.  BA_ESTATE before the first iteration,
 * BA_ENUMERIC if either is non-finite.  Host pointers. */
int ba_bounds(ba_ctx *c, double *I_lower, double *maxD_upper);

/* Copy p (2^n doubles) to a host buffer.  Synchronises. */
int ba_get_p(ba_ctx *c, double *p_host);

/* ---- forced additions ------------------------------------------------------------ */

/* Bytes of device scratch ba_create_ext needs for size n (0 if n is invalid). */
size_t ba_scratch_bytes(int n);

/* As ba_create, on caller-owned DEVICE buffers: p_dev (2^n doubles), q_dev (2^{n+1}-1 doubles),
 * D_dev (2^n doubles), scratch_dev (>= ba_scratch_bytes(n), 256-byte aligned) and a cudaStream_t
 * passed as void* (NULL = legacy default stream).  p_dev is overwritten with the uniform start. */
int ba_create_ext(int n, double d, void *p_dev, void *q_dev, void *D_dev,
                  void *scratch_dev, size_t scratch_bytes, void *cuda_stream, ba_ctx **out);

/* Switch the context to the paper's EXACT deletion channel BDC_{n,k}:
 * W(y|x) = emb(y,x) / C(n,k) for |y| = k and 0 for every other length, 0 <= k <= n.  The same kernels run
 * with the weight vector w_j = [j = k] / C(n,k); the ENUM sweeps skip the nodes / output prefixes that cannot reach
 * length k (they would only add exact zeros) and enumerate every |z| of the others (the other lengths carry weight 0
 * and q is 0 there).  ba_bounds then brackets C_{n,k}; Lemma 2 combines them into a bound on
 * C_n(d) (harness: python -m paper_2604_05867_b200.exact).  Only before the first iteration: BA_ESTATE otherwise;
 * BA_EINVAL for a bad k. */
int ba_set_exact(ba_ctx *c, int k);

/* Complement symmetry (the cpl half of Theorem 4): emb(cpl y, cpl x) = emb(y, x), so
 * an iterate with p(x) = p(~x) for every x keeps that property, and q(~y) = q(y), D(~x) = D(x).  With on = 1 the ENUM
 * sweeps enumerate only the inputs and the output prefixes whose first symbol is 0 and mirror the results (half the
 * terms per iteration; identical q, D, p up to rounding order of the reductions).  Requires n >= 9 and the current p
 * to be complement-symmetric bit for bit (the uniform start is); ba_set_p then rejects asymmetric vectors.
 * Only in BA_MODE_ENUM: FAST iterations sum D(x) and D(~x) in different orders, so they would break the bit-for-bit
 * symmetry the ENUM sweeps rely on; ba_set_mode(FAST) is refused (BA_EINVAL) while symmetry is on, and
 * ba_set_symmetry(1) is refused in FAST mode.  BA_EINVAL otherwise. */
int ba_set_symmetry(ba_ctx *c, int on);

/* Select BA_MODE_ENUM (default) or BA_MODE_FAST for subsequent iterations.  BA_EINVAL for an unknown mode, or for
 * FAST while complement symmetry is on. */
int ba_set_mode(ba_ctx *c, int mode);

/* Replace p by a host vector (2^n doubles).  Rejects non-finite or non-positive entries and
 * |sum p - 1| > 1e-9; stores the values as given, without renormalising.  Synchronises. */
int ba_set_p(ba_ctx *c, const double *p_host);

/* q_{K-1} (2^{n+1}-1 doubles) and D_{K-1} (2^n doubles) to host.  BA_ESTATE before any iteration. */
int ba_get_q(ba_ctx *c, double *q_host);
int ba_get_D(ba_ctx *c, double *D_host);

/* log2 Z of the last iteration (the paper's stop statistic is U - log2 Z) and the number
 * of iterations done on this ctx.  Either pointer may be NULL.  Synchronises. */
int ba_stats(ba_ctx *c, double *log2Z, long long *iters_done);

/* History of the last `count` iterations, oldest first: out[3*i+0..2] = {I_t, U_t, log2 Z_t}.
 * count must not exceed min(iters_done, 65536).  Synchronises. */
int ba_get_history(ba_ctx *c, int count, double *out_host);

/* Device-side time of the four phases of the most recent ba_iterate call, averaged per iteration, in
 * milliseconds, measured with CUDA events on the ctx stream: ms[0] output sweep, ms[1] input sweep,
 * ms[2] reductions + update, ms[3] whole iteration.  Only the LAST 64 iterations of the call are timed (a call of
 * k > 64 iterations reports the average over its last 64).  BA_ESTATE before the first iteration.  Synchronises. */
int ba_last_timing(ba_ctx *c, double ms_host[4]);

/* Device-side time, in milliseconds, of the one-off set-up pass that the first ba_iterate (and the first after
 * ba_set_exact) runs before its iterations: the enumerating pass that builds Hc(x) = sum_y W log2(emb / ebar_k), the
 * iteration-independent half of the hoisted logarithm.  BA_ESTATE before it ran.  Synchronises. */
int ba_setup_ms(ba_ctx *c, double *ms_host);

/* Microbenchmarks of the pipes the ENUM sweeps are bound by, on the current device (no ctx needed; default stream;
 * synchronises the device; a few milliseconds): out[0] FP64 FMA, out[1] IDP.2A (the integer multiply pipe), out[2]
 * conflict-free LDS.64, out[3] FP32 FMA (= issue rate), each in warp-instructions per clock per SM; out[4] SM clock in
 * MHz seen by the kernels; out[5] number of SMs.  SURVEY 8(d): the roofline denominators are measured in the same run
 * as the number they divide.  Host pointer. */
int ba_measure_peaks(double out_host[6]);

/* Row x of the integer embedding matrix as produced by the input-sweep enumerator:
 * emb_out_host[idx(y)] = emb(y,x) for every y, zero where y is not a subsequence.  2^{n+1}-1 entries. */
int ba_debug_emb_row(ba_ctx *c, unsigned x, unsigned *emb_out_host);

/* Column yidx of the embedding matrix as produced by the output-sweep supersequence enumerator
 * (P:240): emb_out_host[x] = emb(y,x).  2^n entries. */
int ba_debug_emb_col(ba_ctx *c, unsigned yidx, unsigned *emb_out_host);

/* Number of (x,y) terms T(n) = sum_k 2^k sum_{i<=n-k} C(n,i) (Lemma 6) visited by one sweep,
 * and, after ba_debug_count_terms, the number the ENUM input / output enumerators actually visited
 * (device-side integer checksums).  Host pointers. */
int ba_terms_per_sweep(int n, unsigned long long *T);
int ba_debug_count_terms(ba_ctx *c, unsigned long long *in_terms, unsigned long long *out_terms,
                         unsigned long long *in_emb_sum, unsigned long long *out_emb_sum);

/* Host-only self-check of the static pair tables the ENUM kernels use for a low tile of m bits (1 <= m <= 8;
 * m = min(n, 8)): under each of the 16 classes every pair (v, z) -- v in {0,1}^m, z a non-empty subsequence of
 * v -- must be served exactly once, by a fast pair or by a rider, with the embedding counts B(sigma_s.z, v)
 * an independent DP gives.  stats[0] / stats[2] = fast pairs of the input / output tables summed over
 * the classes, stats[1] / stats[3] = riders; so stats[0] + stats[1] = stats[2] + stats[3] = 16 (T(m) - 2^m)
 * (Lemma 6).  Needs no device.  Returns BA_OK or BA_EINVAL.  Host pointer. */
int ba_debug_check_tables(int m, unsigned long long stats[4]);

void ba_destroy(ba_ctx *c);
const char *ba_last_error(const ba_ctx *c);

/* ---- no-allocation entry point ------------------------------------------------------------------ */

/* For callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it): the epilogue of the input sweep without a ctx.  D(x) = Hc(x) - (S0(x) + S1(x)) for the 2^n inputs
 * (S1_dev may be NULL: D = Hc - S0), and the reductions of the bounds and of the update:
 *     out3 = { sum_x p(x) D(x),  max_x D(x),  sum_x p(x) 2^D(x) }   (= I_t, U_t, Z_t of ba_bounds / ba_stats).
 * All pointers are DEVICE pointers to float64, caller-owned: Hc, S0, S1, p of 2^n entries (read), D of 2^n entries
 * and out3 of 3 entries (written).  The two kernels are queued on `stream` (a cudaStream_t, NULL = the default
 * stream) of the CURRENT device; the call does not synchronise and copies nothing to the host.
 *
 * The first-stage partial sums live in a file-scope device array of the library (BA_NOALLOC_MAXBLK triples = 48 KB,
 * held by every GPU that loads libba until the process exits) instead of ctx scratch, so the call performs no
 * cudaMalloc / cudaFree and calls no allocating routine; the first call on a device only looks up the array's device
 * address.  Limit: n <= BA_NOALLOC_NMAX (one block partial per 2^15 inputs); beyond it BA_EINVAL, nothing is launched,
 * and ba_noalloc_last_error() says why.  Every call on a device shares the array, which keeps the last call's
 * contents: a call overwrites every entry it later reads (nothing has to be cleared), and two calls that overlap on
 * the GPU (different streams, or concurrent graph branches) race on it -- serialise them.  Sums are formed in a
 * fixed order: results are bit-reproducible for a given n. */
#define BA_NOALLOC_MAXBLK 2048
#define BA_NOALLOC_NMAX 26
int ba_in_final_noalloc(int n, const void *Hc_dev, const void *S0_dev, const void *S1_dev, const void *p_dev,
                        void *D_dev, void *out3_dev, void *stream);
/* Message of the calling thread's last failed ba_in_final_noalloc ("" after a success).  Static storage. */
const char *ba_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* BA_H */
