/*
 * sparse_attn.h -- C ABI of the B200 (sm_100a) tile-skipping attention forward pass.
 *
 * One hot path of arxiv/paper_2606_16317 ("Training-Free Sparse Attention Based on Cumulative
 * Energy Filtering"): a FlashAttention-style forward pass for non-causal self-attention that
 * decides, inside the K-tile loop and from the online-softmax statistics only, whether a
 * (Q_i, K_j) tile is skipped (section 3.1, Eq. 5-6).  No mask pre-pass.
 *
 * All entry points are plain C, never throw, never exit the process, and allocate no persistent
 * device memory (the one fixed exception is the 16 MiB static array behind
 * sparse_attn_row_topk_curve_static, which is part of the library's device image).  There is no
 * CPU fallback: on a machine without an sm_100 device every compute call fails with
 * SPARSE_ATTN_ERR_DEVICE.
 */
#ifndef SPARSE_ATTN_H_
#define SPARSE_ATTN_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPARSE_ATTN_VERSION 100 /* 0.1.0 */

/* mode argument of sparse_attn_fwd */
enum sparse_attn_mode {
    SPARSE_ATTN_DENSE = 0,   /* no skipping: softmax(scale * Q K^T) V, FlashAttention-2 tiling */
    SPARSE_ATTN_FIXED = 1,   /* BLASST-style: skip tile j iff  mhat_r - m_r^(j-1) < lambda  for every valid row r
                                (tile max minus running max over retained tiles) */
    SPARSE_ATTN_DYNAMIC = 2, /* DynSparse: skip tile j iff  t_r = mhat_r - LSE_r^(j-1) < lambda  for every valid row r,
                                LSE over the retained tiles only (Eq. 5-6) */
    SPARSE_ATTN_MASK = 3     /* mask-driven: the decisions are READ from params->skip_mask_in instead of being taken in the
                                loop -- the block-mask methods the paper compares with (Top-K, Top-P, the "ideal" mask of
                                section 3; Fig. 3) run through the same kernel.  Everything else
                                is as in the other sparse modes: retained tiles only enter m, l, O and lse (Eq. 1, Eq. 6).
                                Tile j = 0 of every row of tiles is retained whatever its byte says. */
};

/* return codes: 0 on success, negative on error */
enum sparse_attn_status {
    SPARSE_ATTN_OK = 0,
    SPARSE_ATTN_ERR_NULL_POINTER = -1, /* a required pointer is NULL */
    SPARSE_ATTN_ERR_SHAPE = -2,        /* B, H or N <= 0, or B*H / N too large for the launch */
    SPARSE_ATTN_ERR_HEAD_DIM = -3,     /* D not in {64, 128} */
    SPARSE_ATTN_ERR_TILE = -4,         /* tile_q / tile_k not a supported decision tile for this D and mode */
    SPARSE_ATTN_ERR_MODE = -5,         /* mode not in {0, 1, 2, 3} */
    SPARSE_ATTN_ERR_PARAMS = -6,       /* params NULL in a sparse mode, struct_size wrong, lambda NaN,
                                          lambda > 0 in FIXED mode or with tile_k < 128 at D = 128, softmax_scale
                                          negative / non-finite, skip_mask_in NULL in MASK mode or set in another mode */
    SPARSE_ATTN_ERR_ALIGNMENT = -7,    /* q, k, v or out not 16-byte aligned (TMA / vector stores) */
    SPARSE_ATTN_ERR_DEVICE = -8,       /* no CUDA device, or the current device is not sm_100 (B200) */
    SPARSE_ATTN_ERR_CUDA = -9          /* a CUDA runtime / driver call failed; see sparse_attn_last_error() */
};

/*
 * Threshold and launch parameters.  Host struct, plain C; the first field versions it.
 */
typedef struct sparse_attn_params {
    uint32_t struct_size;   /* must be sizeof(sparse_attn_params) */
    float lambda;           /* threshold lambda of PAPER.md:123, natural-log logit units (S includes the softmax
                               scale).  A tile is skipped iff max over its valid rows of t_r is < lambda (strict).
                               -INFINITY disables skipping.  In FIXED mode it is ln(alpha) and must be <= 0. */
    float softmax_scale;    /* 0 means 1/sqrt(D) */
    int32_t tile_q;         /* decision tile rows B_r; 0 = default (64 for D = 64, 128 for D = 128) */
    int32_t tile_k;         /* decision tile columns B_c; 0 = default (same as tile_q).
                               D = 128 also accepts tile_q = 128 with tile_k = 64 or 32 in the sparse modes ("block
                               size 32"): the decision tiles of 64 / 32 keys are visited in ascending
                               key order, the statistics are updated after every retained one, and exp, row sum and
                               P V are skipped per decision tile.  T_c below is then ceil(N / tile_k).  With these
                               narrow tiles lambda must be <= 0 (the softmax stabiliser follows the max of the whole
                               128-key MMA tile, which only a non-positive threshold is certain to retain). */
    void* stream;           /* cudaStream_t to launch on; NULL = the default stream */
    uint8_t* skip_mask_out; /* optional, device, [B, H, T_r, T_c] bytes, 1 = tile skipped, fully overwritten.
                               T_r = ceil(N / tile_q), T_c = ceil(N / tile_k).  NULL in timed runs. */
    float* margin_out;      /* optional, device, [B, H, T_r, T_c] fp32: g_ij = max_r t_r - lambda as evaluated on
                               the GPU (+inf for tile 0 and in DENSE mode; in MASK mode the DYNAMIC margin of the state
                               the mask built).  Debug / parity only. */
    const uint8_t* skip_mask_in; /* MASK mode only (must be NULL otherwise): device, [B, H, T_r, T_c] bytes, non-zero =
                               skip the tile; never written.  Default decision tiles only (tile_q = tile_k = default). */
    uint64_t* cycles_out;   /* optional, device, uint64[2], overwritten: {sum over the CTAs of the launch of the SM clock
                               cycles (clock64) each CTA ran, number of CTAs}.  With one CTA resident per SM and a grid of
                               whole waves, sum / (SM count * kernel time) is the SM clock the launch actually ran at --
                               measurement support (bench.py), selects the debug instantiation of the kernel; not
                               supported by sparse_attn_fwd_host (must be NULL there). */
} sparse_attn_params;

/*
 * Forward pass.  Enqueues work on params->stream (or the default stream) and returns; the caller
 * synchronises.  One GPU, the current device.
 *
 *   q, k, v  device, bf16, [B, H, N, D] contiguous, 16-byte aligned, never written
 *   out      device, bf16, [B, H, N, D]; fully overwritten.  Rows are renormalised over the retained
 *            tiles (Eq. 1): out_r = sum_{c in retained tiles} e^{S_rc - lse_r} v_c
 *   lse      device, fp32, [B, H, N], natural log, over the retained tiles (Eq. 6); may be NULL
 *   B,H,N,D  batch, heads, tokens (N_q = N_k, non-causal), head dim in {64, 128}
 *   params   host pointer; may be NULL only when mode == SPARSE_ATTN_DENSE
 *   mode     enum sparse_attn_mode
 *   stats_out device, int64, [B, H, 2] = {executed, skipped} decision-tile counts per head
 *            (executed + skipped = T_r * T_c; "Sps"); overwritten; may be NULL
 *
 * K tiles are visited in ascending token order for every Q tile (decisions are order dependent);
 * tile j = 0 is never skipped; a skipped tile leaves m, l and O untouched; Q K^T is computed for
 * every tile, exp / row-sum / P V only for retained ones.
 *
 * Returns SPARSE_ATTN_OK or a negative sparse_attn_status; arguments are validated on the host
 * before anything is launched, so on error nothing has been written.
 */
int sparse_attn_fwd(const void* q, const void* k, const void* v, void* out, float* lse,
                    int B, int H, int N, int D,
                    const sparse_attn_params* params, int mode, int64_t* stats_out);

/*
 * Same operation with HOST buffers (pinned for full speed; pageable works, without overlap): cuts
 * the B*H heads (independent units) into up to 20 chunks and pipelines them over four internal
 * streams -- the host->device copy of chunk c+1 and the device->host copy of chunk c-1 run under the
 * kernel of chunk c, consecutive kernels alternate between two streams -- then synchronises.
 * params->skip_mask_out / margin_out / skip_mask_in, if set, are host pointers here too; work is
 * ordered after whatever is already enqueued on params->stream.  Used for end-to-end timing;
 * layouts as above.  Synchronous: on return every output buffer is complete.
 * Memory: the device copies of q, k, v, out (and of the optional buffers) come from a stream-ordered
 * memory pool that belongs to this library (one per device; the device's default pool and its
 * attributes are never touched).  Freed scratch STAYS in that pool for the next call -- after a
 * config-3-sized call about 4 GB -- until sparse_attn_release_scratch() returns it to the driver.
 * The internal streams and events are recycled across calls in the same way.
 */
int sparse_attn_fwd_host(const void* q, const void* k, const void* v, void* out, float* lse,
                         int B, int H, int N, int D,
                         const sparse_attn_params* params, int mode, int64_t* stats_out);

/* Returns the memory that sparse_attn_fwd_host keeps in the library's scratch pool of the CURRENT device to the
 * driver (cudaMemPoolTrimTo 0) and destroys that device's recycled internal streams / events.  Call it when no
 * sparse_attn_fwd_host call is running on the device; the next such call simply allocates again. */
int sparse_attn_release_scratch(void);

/* lambda = ln((1 - recall) / N): the worst-case threshold under which every row keeps more than
 * `recall` of its softmax mass (lambda = ln(eps / L)).  Pure host function. */
double sparse_attn_lambda_from_recall(double recall, int N);

/* lambda = ln(p_real) + ln(tile_k / N)  (Eq. 7).  Pure host function. */
double sparse_attn_lambda_from_preal(double p_real, int tile_k, int N);

/*
 * Spatio-temporal token re-ordering around the kernel (last sentence: "mapping the one-dimensional
 * sequence back to its original spatiotemporal dimensions before processing ... can enhance the correlation within
 * tiles"; PAPER.md:25 names the technique).  Tokens of a [grid_t, grid_h, grid_w] latent grid, stored in
 * [t, h, w] order (n = (t * grid_h + h) * grid_w + w), are regrouped into bricks of brick_t x brick_h x brick_w
 * cells so that 128 consecutive tokens are neighbours in time and space.
 *
 * sparse_attn_brick_permutation: pure host function.  Writes perm_out[p] = n, the original index of the token at
 * position p of the brick order: bricks are visited in (t, h, w) order of their origin, the cells of a brick in
 * (t, h, w) order; bricks at the upper edges of the grid are clipped to it (no padding), so perm_out is a
 * permutation of 0 .. N-1 with N = grid_t * grid_h * grid_w.  perm_out is HOST memory, N int32, caller-owned.
 * Errors: NULL pointer, any dimension <= 0, or N > 2^24 (SPARSE_ATTN_ERR_SHAPE).
 */
int sparse_attn_brick_permutation(int grid_t, int grid_h, int grid_w, int brick_t, int brick_h, int brick_w,
                                  int32_t* perm_out);

/*
 * sparse_attn_reorder_tokens: gathers (inverse = 0) or scatters (inverse = 1) the token rows of a bf16 [B, H, N, D]
 * tensor on the device:
 *     inverse = 0:  dst[b, h, p, :]       = src[b, h, perm[p], :]     (into brick order, before the attention call)
 *     inverse = 1:  dst[b, h, perm[p], :] = src[b, h, p, :]           (back to [t, h, w] order, on the output)
 * src, dst: DEVICE, contiguous, 16-byte aligned, must not overlap; perm: DEVICE, N int32, a permutation of 0 .. N-1.
 * Row-wise attention is permutation-equivariant: running sparse_attn_fwd on re-ordered q, k, v and scattering `out`
 * back gives, in DENSE mode, the result of the un-permuted call up to summation order; in the sparse modes the
 * decisions are taken on the re-ordered tiles (that is the point).  HBM-bound: 2 * B*H*N*D*2 bytes per call.
 * Enqueues one kernel on `stream` (cudaStream_t, NULL = default stream) and returns; no host synchronisation.
 * The entries of perm are NOT validated on the device (an out-of-range entry is undefined behaviour, as for any
 * index array handed to a gather); sparse_attn_brick_permutation always produces a valid one.
 * Errors: NULL pointers, bad shape, D not in {64, 128}, misaligned or overlapping buffers, no sm_100 device.
 */
int sparse_attn_reorder_tokens(const void* src, void* dst, int B, int H, int N, int D, const int32_t* perm,
                               int inverse, void* stream);

/*
 * Block mass of the dense attention probabilities (the quantity block-level Top-K / Top-P selection ranks,
 * PAPER.md:61-62, and the "softmax ... before FA" of section 3):
 *     mass_out[b, h, i, j] = sum over the rows r of Q tile i and the columns c of K tile j of  e^{S_rc - lse[b, h, r]}
 * with S = softmax_scale * Q K^T and lse the DENSE log-sum-exp of row r (as sparse_attn_fwd returns it in DENSE
 * mode), so that every row of tiles sums to the number of valid rows of Q tile i.  The Q K^T pipeline of the forward
 * kernel without P V (one pass over all tiles, tensor cores + one ex2 per logit).
 *   q, k     device, bf16, [B, H, N, D] contiguous, 16-byte aligned        lse   device, fp32, [B, H, N]
 *   mass_out device, fp32, [B, H, T, T] with T = ceil(N / tile), tile = 64 (D = 64) or 128 (D = 128); overwritten
 *   softmax_scale  0 means 1/sqrt(D);   stream  cudaStream_t, NULL = default.  Enqueues and returns.
 * Sums are fp32 atomics: the result is reproducible to rounding, not bit for bit.
 */
int sparse_attn_block_mass(const void* q, const void* k, const float* lse, float* mass_out, int B, int H, int N, int D,
                           float softmax_scale, void* stream);

/*
 * sparse_attn_block_mass plus the per-tile sum of SQUARED probabilities, the other ingredient of the error-variance
 * bound of Eq. 2-3 (Var(E) = sigma^2 [sum_S p_j^2 + (S_1/(1-S_1))^2 sum_K p_j^2]):
 *     sqmass_out[b, h, i, j] = sum over the rows r of Q tile i and the columns c of K tile j of  e^{2 (S_rc - lse[b, h, r])}
 * Same pass, same layout and arguments as sparse_attn_block_mass; sqmass_out may be NULL (then identical to it).
 */
int sparse_attn_block_stats(const void* q, const void* k, const float* lse, float* mass_out, float* sqmass_out,
                            int B, int H, int N, int D, float softmax_scale, void* stream);

/*
 * Block selectors on a block-mass matrix (the comparison methods of PAPER.md:61-62, Table 1, Fig. 3), producing the
 * bitmap SPARSE_ATTN_MASK consumes.  Per row of tiles (b, h, i):
 *   SPARSE_ATTN_SELECT_TOPK  retain the ceil(param * T_c) tiles of largest mass (a fixed budget; param = kept fraction)
 *   SPARSE_ATTN_SELECT_TOPP  retain tiles in order of decreasing mass until their share of the row's total mass reaches
 *                            param (the tile that crosses it is retained)
 * Equal masses are ordered by the lower tile index first; tile 0 is always retained.  param in (0, 1].
 *   mass          device, fp32, [B, H, T_r, T_c] (sparse_attn_block_mass)     T_c <= 4096
 *   skip_mask_out device, bytes, [B, H, T_r, T_c], 1 = skip; fully overwritten
 * An offline analysis step (O(T_c^2) per row of tiles), enqueued on `stream`.
 */
enum sparse_attn_selector { SPARSE_ATTN_SELECT_TOPK = 0, SPARSE_ATTN_SELECT_TOPP = 1 };
int sparse_attn_select_blocks(const float* mass, uint8_t* skip_mask_out, int B, int H, int T_r, int T_c, int kind,
                              double param, void* stream);

/*
 * The "ideal" mask of PAPER.md section 3 (lines 105-109) at block level, for SPARSE_ATTN_MASK: "Given an upper
 * tolerance limit for the error variance Theta ... sort P_j in ascending order ... sequentially move the smallest
 * p_j from K to S ... stop when the condition represented by Eq. 3 is met".  Per row of tiles (b, h, i), with
 * P_j = mass[i, j] / rows_i and q_j = sqmass[i, j] / rows_i (block sums averaged over the rows_i valid rows of Q tile i):
 * tiles j >= 1 are discarded in order of increasing mass (equal masses: lower index first) for as long as
 *     sum_{S} q_j + (S_1 / (1 - S_1))^2 * sum_{K} q_j <= theta,        S_1 = sum_{S} P_j            (Eq. 3)
 * holds with the tile included in S; the scan stops at the first tile that would violate it.  Tile 0 is never a
 * candidate (MASK mode retains it regardless).  theta = 0 discards only tiles of zero mass.
 *   mass, sqmass   device, fp32, [B, H, T_r, T_c] (sparse_attn_block_stats);  T_r = ceil(N / tile_q), T_c <= 4096
 *   skip_mask_out  device, bytes, [B, H, T_r, T_c], 1 = skip; fully overwritten
 *   N, tile_q      tokens and decision-tile rows (64 or 128): rows_i = min(tile_q, N - i * tile_q)
 * "Requires softmax computation, sorting, and dynamic decision-making before FA": an offline
 * comparison method, O(T_c^2) per row of tiles, enqueued on `stream`.
 */
int sparse_attn_select_blocks_greedy(const float* mass, const float* sqmass, uint8_t* skip_mask_out, int B, int H, int N,
                                     int tile_q, int T_c, double theta, void* stream);

/*
 * Quality of a sparse run against the dense run of the same inputs, reduced on the device (harness support; the
 * paper's quality measures: recall = kept share of the softmax mass, and |O - O'|).
 *
 * sparse_attn_recall_stats: recall_r = e^{lse_retained[r] - lse_dense[r]} for n_rows rows (both device fp32, natural
 *   log, as sparse_attn_fwd writes them); stats_out (DEVICE, double[2]) = {min_r recall_r, sum_r recall_r}.
 * sparse_attn_output_error: stats_out (DEVICE, double[2]) = {max |a - b|, sum |a - b|} over n_elems bf16 elements
 *   (n_elems even, buffers 4-byte aligned), e.g. a sparse output against the dense one.
 * Each enqueues two small kernels on `stream` and returns; the caller synchronises before reading stats_out.
 */
int sparse_attn_recall_stats(const float* lse_retained, const float* lse_dense, int64_t n_rows, double* stats_out, void* stream);
int sparse_attn_output_error(const void* out_a, const void* out_b, int64_t n_elems, double* stats_out, void* stream);

/*
 * Row-level accuracy-vs-recall analysis of Appendix A.1 ("We sample random rows from the P matrix and
 * apply Top-K with different K values to ablate the recall rate.  Excess Kurtosis is used to measure the 'tailedness'
 * of a data distribution"; Fig. 4, Table 3).  For each sampled query row (bh, r), over ALL N keys of head bh:
 *     p = softmax(softmax_scale * q_r K^T);   kurtosis = m4 / m2^2 - 3 (population moments of the N values of p);
 *     for each K = keep_counts[i]: Top-K = the keys with p >= the K-th largest p (ties at the K-th value are all retained),
 *     recall = sum_TopK p,  O' = sum_TopK p v / recall (Eq. 1),  MAE = mean_d |O_d - O'_d|, O = sum p v.
 *   q, k, v        device, bf16, [B, H, N, D] contiguous, 16-byte aligned
 *   rows           HOST, int32 [n_rows][2] = (b * H + h, r); n_rows <= 2^20      keep_counts  HOST, int32 [n_keep], 1 <= K <= N
 *   kurtosis_out   device, fp64 [n_rows] (NaN for a constant row)
 *   recall_out, mae_out   device, fp64 [n_rows][n_keep]
 *   softmax_scale  0 means 1/sqrt(D);   stream  cudaStream_t, NULL = default
 * One CTA per sampled row; logits and exponentials in fp32, sums and moments in fp64; the K-th largest value is found
 * exactly (bitwise radix select), no sort.  Allocates n_rows * N * 4 bytes of scratch from the stream-ordered pool,
 * copies rows / keep_counts (synchronising `stream` once), enqueues one kernel and returns.  An offline analysis tool.
 * Errors: NULL pointers, bad shape, D not in {64, 128}, a row or K out of range, misaligned buffers, no sm_100 device.
 */
int sparse_attn_row_topk_curve(const void* q, const void* k, const void* v, int B, int H, int N, int D, float softmax_scale,
                               const int32_t* rows, int n_rows, const int32_t* keep_counts, int n_keep,
                               double* kurtosis_out, double* recall_out, double* mae_out, void* stream);

/*
 * sparse_attn_row_topk_curve for callers that must not allocate device memory.
 *
 * Who needs it: a host program that has already given the whole GPU to another allocator (an inference server that
 * reserves all free HBM for its cache at start-up, so that a later cudaMalloc / cudaMallocAsync simply fails with
 * out-of-memory), or one whose request path is forbidden to touch the driver's allocator because cudaMalloc and
 * cudaFree may stall every stream of the device.  sparse_attn_row_topk_curve above takes n_rows * N * 4 bytes plus two
 * small index buffers from the stream-ordered pool on every call; this entry point takes nothing: it calls no
 * cudaMalloc*, no cudaFree* and no library routine that allocates.
 *
 * Same computation, same kernel, same arguments and same results as sparse_attn_row_topk_curve (q, k, v and the three
 * outputs are the caller's device buffers, rows / keep_counts the caller's host arrays).  The only difference is where the
 * kernel's working memory lives: one fixed array inside the library's device image,
 *     SPARSE_ATTN_STATIC_SCRATCH_FLOATS fp32 (16 MiB: one line of N exponentials per sampled row)
 *     + SPARSE_ATTN_STATIC_MAX_ROWS (bh, r) pairs + SPARSE_ATTN_STATIC_MAX_KEEP keep counts  (32 KiB),
 * which every GPU that loads this library holds from the moment its code is loaded until the process exits.
 * Limits, checked before anything is enqueued (SPARSE_ATTN_ERR_SHAPE, nothing written):
 *     (int64) n_rows * N <= SPARSE_ATTN_STATIC_SCRATCH_FLOATS,  n_rows <= SPARSE_ATTN_STATIC_MAX_ROWS,
 *     n_keep <= SPARSE_ATTN_STATIC_MAX_KEEP     (e.g. 128 rows at N = 32760, 55 rows at N = 75600; split larger samples
 *     into several calls, one after the other).
 * Set-up: the first call on each device (made with that device current) looks up the array's device address once and
 * remembers it; make that first call before any stream capture begins.  Later calls on the device do no set-up.
 * Sharing: there is ONE array per device and every call uses it.  Two calls whose kernels may overlap on the GPU (two
 * streams, or two host threads) corrupt each other's results -- run them in stream order or serialise them yourself.
 * The array keeps the previous call's contents; that is harmless here, because each call overwrites the row list, the K
 * list and every element of its rows' lines before anything reads them, so nothing has to be cleared between calls.
 * Like sparse_attn_row_topk_curve it copies rows / keep_counts to the device, synchronises `stream` once (so the caller
 * may reuse them), enqueues one kernel and returns; the caller synchronises before reading the outputs.
 * Errors: those of sparse_attn_row_topk_curve, plus SPARSE_ATTN_ERR_SHAPE beyond the limits above.
 */
#define SPARSE_ATTN_STATIC_SCRATCH_FLOATS (4u << 20)
#define SPARSE_ATTN_STATIC_MAX_ROWS 2048
#define SPARSE_ATTN_STATIC_MAX_KEEP 4096
int sparse_attn_row_topk_curve_static(const void* q, const void* k, const void* v, int B, int H, int N, int D,
                                      float softmax_scale, const int32_t* rows, int n_rows, const int32_t* keep_counts,
                                      int n_keep, double* kurtosis_out, double* recall_out, double* mae_out, void* stream);

/* Static string for a status code. */
const char* sparse_attn_status_string(int status);

/* Detail of the last error on this thread ("" if none).  Valid until the next call on the thread. */
const char* sparse_attn_last_error(void);

/* SPARSE_ATTN_VERSION of the loaded library. */
int sparse_attn_version(void);

/* Number of kernel launches sparse_attn_fwd and sparse_attn_reorder_tokens have enqueued in this process
 * (for bench accounting). */
int64_t sparse_attn_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* SPARSE_ATTN_H_ */
