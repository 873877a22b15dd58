/*
 * dynsparse_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle for the hot path of arxiv/paper_2606_16317
 * ("Training-Free Sparse Attention Based on Cumulative Energy Filtering"): FlashAttention-style
 * forward attention with in-loop tile skipping.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this file.  It shares
 * no code with paper_2606_16317_b200/ (the CUDA path) and is never used as a fallback.
 *
 * What it computes, step by step in the paper's order and notation (section 3.1):
 *
 *   S_rc      = scale * sum_d q_rd k_cd                    logits "A_i"; scale: DESIGN.md G1
 *   mhat_rj   = max_{c in tile j} S_rc                     "local maximum value of each tile"
 *   tau_rj    = ln sum_{c in tile j} e^{S_rc}              energy of tile j (summand of Eq. 6)
 *   DYNAMIC:  t_rj = mhat_rj - LSE_r^(j-1)                 Eq. 5
 *   FIXED:    t_rj = mhat_rj - m_r^(j-1)                   BLASST indicator (R6)
 *   skip tile (i,j)  iff  max_r t_rj < lambda              PAPER.md:123, strict "<"; all-rows reading DESIGN.md R1
 *   kept:     LSE_r <- ln(e^{LSE_r} + e^{tau_rj}),  m_r <- max(m_r, mhat_rj)      Eq. 6, sum over k not in J_i
 *   skipped:  state untouched                              Eq. 6 (k notin J_i)
 *   tile j=0 is always kept (LSE^(0) = -inf, t = +inf)     DESIGN.md R3
 *   O_r       = sum_{c in retained tiles} e^{S_rc - LSE_r} v_c    renormalised over the kept set, Eq. 1
 *   lse_r     = LSE_r (natural log, over retained tiles)
 *
 * Dense mode keeps every tile, so O is softmax(scale * Q K^T) V by definition.
 *
 * Each Q tile is independent; they are run in parallel with OpenMP, nothing else is blocked,
 * fused or reordered.  Inputs are bf16 bit patterns, widened exactly to fp64.
 *
 * Pins (tests/test_oracle_pins.py): P1 dense == textbook softmax / torch fp64 SDPA; P2/P3 recall
 * bound; P4 counts; P5 Eq. 1 identity; P6 DYNAMIC superset of FIXED; P7-P9 closed forms; P10 brute force --
 * P7-P10 also with rectangular decision tiles (tile_k != tile_q: 128 x 32, 128 x 64, 64 x 16).
 * Parity unpinned: the absolute sparsity reached on any input (the paper's 61-82 % are on Wan 2.2
 * activations, which are not available).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { MODE_DENSE = 0, MODE_FIXED = 1, MODE_DYNAMIC = 2 };

static double bf16_to_f64(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* ln(e^a + e^b) with -inf handled (a = -inf before the first retained tile). */
static double logaddexp(double a, double b) {
    if (a == -INFINITY) return b;
    if (b == -INFINITY) return a;
    double hi = a > b ? a : b, lo = a > b ? b : a;
    return hi + log1p(exp(lo - hi));
}

/* S_rc for one (row, column): scale * sum_d q_rd k_cd, d ascending. */
static double logit(const double* q, const double* k, int D, int r, int c, double scale) {
    double acc = 0.0;
    for (int d = 0; d < D; ++d) acc += q[(size_t)r * D + d] * k[(size_t)c * D + d];
    return scale * acc;
}

int dynsparse_oracle_version(void) { return 1; }

int dynsparse_oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * One head.  q, k, v: bf16 bits, [N, D] row-major.
 * qtiles: indices of the Q tiles to run (NULL: all T_r tiles, n_qtiles must then be T_r).
 * forced_skip: NULL for a free run.  Otherwise [n_qtiles, T_c] and the oracle *replays* that
 *   bitmap (1 = skipped): it follows the given decisions but still evaluates the margin g_ij
 *   from the state built by the tiles the bitmap kept (SURVEY.md section 8(c) "replay").
 * Outputs (all caller-allocated):
 *   out    [n_qtiles, tile_q, D] fp64, rows beyond N are zero
 *   lse    [n_qtiles, tile_q]    fp64 (0 for rows beyond N)
 *   skip   [n_qtiles, T_c]       1 = skipped (free run: the oracle's decision; replay: copy of forced)
 *   margin [n_qtiles, T_c]       g_ij = max_r t_rj - lambda; +inf where t is +inf (first retained tile) or mode DENSE
 * Returns 0, or -1 on a bad argument.
 */
int dynsparse_oracle_head(const uint16_t* q_bits, const uint16_t* k_bits, const uint16_t* v_bits,
                          int N, int D, int tile_q, int tile_k, double scale, double lambda, int mode,
                          const int32_t* qtiles, int n_qtiles, const uint8_t* forced_skip,
                          double* out, double* lse, uint8_t* skip, double* margin, int n_threads) {
    if (!q_bits || !k_bits || !v_bits || !out || !lse || !skip || !margin) return -1;
    if (N <= 0 || D <= 0 || tile_q <= 0 || tile_k <= 0 || mode < 0 || mode > 2) return -1;
    const int T_r = (N + tile_q - 1) / tile_q, T_c = (N + tile_k - 1) / tile_k;
    if (!qtiles && n_qtiles != T_r) return -1;

    double* q = (double*)malloc(sizeof(double) * (size_t)N * D);
    double* k = (double*)malloc(sizeof(double) * (size_t)N * D);
    double* v = (double*)malloc(sizeof(double) * (size_t)N * D);
    if (!q || !k || !v) { free(q); free(k); free(v); return -1; }
    for (size_t i = 0; i < (size_t)N * D; ++i) {
        q[i] = bf16_to_f64(q_bits[i]);
        k[i] = bf16_to_f64(k_bits[i]);
        v[i] = bf16_to_f64(v_bits[i]);
    }
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif

    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int t = 0; t < n_qtiles; ++t) {
        const int i = qtiles ? qtiles[t] : t;
        if (i < 0 || i >= T_r) { bad = 1; continue; }
        const int r0 = i * tile_q;
        const int rows = (N - r0 < tile_q) ? (N - r0) : tile_q;      /* valid rows (R9) */
        double* L = (double*)malloc(sizeof(double) * tile_q);        /* LSE_r over retained tiles, Eq. 6 */
        double* M = (double*)malloc(sizeof(double) * tile_q);        /* m_r over retained tiles */
        for (int r = 0; r < tile_q; ++r) { L[r] = -INFINITY; M[r] = -INFINITY; }
        uint8_t* sk = skip + (size_t)t * T_c;
        double* mg = margin + (size_t)t * T_c;
        const uint8_t* forced = forced_skip ? forced_skip + (size_t)t * T_c : NULL;

        /* pass 1: decisions and the running statistics, K tiles in ascending order (R4) */
        for (int j = 0; j < T_c; ++j) {
            const int c0 = j * tile_k;
            const int cols = (N - c0 < tile_k) ? (N - c0) : tile_k;
            double g = -INFINITY;          /* max_r t_rj - lambda */
            int have_state = 1;
            double* mhat = (double*)malloc(sizeof(double) * rows);
            double* tau = (double*)malloc(sizeof(double) * rows);
            double* S = (double*)malloc(sizeof(double) * (size_t)rows * cols);   /* S_ij, this tile only */
            for (int r = 0; r < rows; ++r)
                for (int c = 0; c < cols; ++c) S[(size_t)r * cols + c] = logit(q, k, D, r0 + r, c0 + c, scale);
            for (int r = 0; r < rows; ++r) {
                double mx = -INFINITY;
                for (int c = 0; c < cols; ++c) if (S[(size_t)r * cols + c] > mx) mx = S[(size_t)r * cols + c];
                double sum = 0.0;
                for (int c = 0; c < cols; ++c) sum += exp(S[(size_t)r * cols + c] - mx);
                mhat[r] = mx;
                tau[r] = mx + log(sum);
                const double ref = (mode == MODE_FIXED) ? M[r] : L[r];
                if (ref == -INFINITY) have_state = 0;   /* nothing retained yet: t = +inf */
                else { double tr = mx - ref; if (tr - lambda > g) g = tr - lambda; }
            }
            free(S);
            if (!have_state || mode == MODE_DENSE) g = INFINITY;
            int do_skip;
            if (forced) do_skip = forced[j] != 0;
            else do_skip = (mode != MODE_DENSE) && (g < 0.0);          /* strict: PAPER.md:123 */
            sk[j] = (uint8_t)do_skip;
            mg[j] = g;
            if (!do_skip) {
                for (int r = 0; r < rows; ++r) {
                    L[r] = logaddexp(L[r], tau[r]);
                    if (mhat[r] > M[r]) M[r] = mhat[r];
                }
            }
            free(mhat); free(tau);
        }

        /* pass 2: O_r = sum over retained columns of e^{S_rc - L_r} v_c  (Eq. 1: renormalised over the kept set) */
        double* o = out + (size_t)t * tile_q * D;
        memset(o, 0, sizeof(double) * (size_t)tile_q * D);
        for (int r = 0; r < tile_q; ++r) lse[(size_t)t * tile_q + r] = (r < rows) ? L[r] : 0.0;
        for (int j = 0; j < T_c; ++j) {
            if (sk[j]) continue;
            const int c0 = j * tile_k;
            const int cols = (N - c0 < tile_k) ? (N - c0) : tile_k;
            for (int r = 0; r < rows; ++r) {
                for (int c = 0; c < cols; ++c) {
                    double p = exp(logit(q, k, D, r0 + r, c0 + c, scale) - L[r]);
                    for (int d = 0; d < D; ++d) o[(size_t)r * D + d] += p * v[(size_t)(c0 + c) * D + d];
                }
            }
        }
        free(L); free(M);
    }
    free(q); free(k); free(v);
    return bad ? -1 : 0;
}
