// Tile-skipping FlashAttention forward for sm_100a (B200).
//
// Implements SURVEY.md section 8(a) steps a1-a9 / PAPER.md section 3.1 in ONE kernel, four modes:
// DENSE, FIXED (BLASST indicator), DYNAMIC (DynSparse, Eq. 5-6) and MASK (decisions
// read from a precomputed block bitmap: the block-mask methods of PAPER.md:61-62 through the same pipeline).
//
// CTA = 2 MMA tiles (slots X = 0, 1) of 128 query rows of one (b, h), sharing every K_j / V_j tile:
//   warps 0-3   softmax warpgroup of slot 0 (thread <-> query row <-> TMEM lane)
//   warps 4-7   softmax warpgroup of slot 1
//   warp  8     TMA producer for Q (once) and the K ring (runs ahead of the decisions)
//   warp  9     tcgen05.mma issuer of slot 0 (of both slots in DENSE mode; one elected lane) and TMEM owner
//   warp  10    TMA producer for the V ring: slot j % NV holds V_j.  DENSE: every tile.  Sparse modes: this warp
//               reads both slots' votes on tile j and fetches V_j only if some slot keeps tile j (plus V_{j+1}
//               speculatively after a kept tile); an unneeded tile completes its ring phase without a load
//   warp  11    tcgen05.mma issuer of slot 1 in the sparse modes (idle in DENSE mode)
// One issuer warp per slot in the sparse modes: a thread that issues tcgen05.mma is held until its last MMA has been dispatched to the
// tensor pipe, so with a single issuer every barrier wait and vote decode of one slot left the pipe idle; with two,
// the control work of one slot overlaps the MMAs of the other.
// TMEM (512 columns): S_0 | S_1 (fp32, BC columns each; P_X, bf16x2, aliases the first BC/2 columns of S_X)
//                     O_0 | O_1 (fp32, D columns each).
// Per slot X and K tile j:  S_X = Q_X K_j^T (always)  ->  softmax warpgroup: row max, skip predicate,
// all-rows vote  ->  skipped: nothing else;  kept: online-softmax update, P_X -> TMEM, O_X += P_X V_j.
// While slot 0 is in its softmax, the tensor pipe works for slot 1 and vice versa.
//
// Decision tiles are BR x BC with BR = 128 / G: G = 1 for the 128 x 128 tiles of D = 128, G = 2 for the
// 64 x 64 tiles of D = 64 (two decision tiles stacked in one M = 128 MMA; a half that skips while its
// partner keeps writes P = 0 and leaves its statistics untouched).
#pragma once
#include "ptx.cuh"

namespace dsa {

#ifdef DSA_PROF
#if DSA_PROF == 2   // timeline of CTA (0, 0) only, no per-phase accumulators
#define PROF_DECL(n)
#define PROF_TICK(i)
#define PROF_FLUSH(base, n, cond)
#else
#define PROF_DECL(n) unsigned long long prof_acc[n] = {}; long long prof_t = clock64();
#define PROF_TICK(i) { long long t__ = clock64(); prof_acc[i] += t__ - prof_t; prof_t = t__; }
#define PROF_FLUSH(base, n, cond) if (a.prof && (cond)) { for (int i__ = 0; i__ < n; ++i__) a.prof[(static_cast<size_t>(blockIdx.y) * gridDim.x + blockIdx.x) * 32 + base + i__] = prof_acc[i__]; }
#endif
#define TRACE(slot) if (a.prof && blockIdx.x == DSA_TRACE_CTA && blockIdx.y == 0 && j >= DSA_TRACE_J0 && j < DSA_TRACE_J0 + 32 && (threadIdx.x & 31) == 0) a.prof[(1 << 20) + ((j - DSA_TRACE_J0) * 2 + x) * 32 + (slot)] = clock64();
#ifndef DSA_TRACE_CTA
#define DSA_TRACE_CTA 0
#endif
#ifndef DSA_TRACE_J0
#define DSA_TRACE_J0 0
#endif
#else
#define TRACE(slot)
#define PROF_DECL(n)
#define PROF_TICK(i)
#define PROF_FLUSH(base, n, cond)
#endif

enum : int { kModeDense = 0, kModeFixed = 1, kModeDynamic = 2, kModeMask = 3,
             kModeMass = 4 };   // internal: block mass of the dense probabilities (sparse_attn_block_mass), no P V

constexpr int kNumThreads = 384;      // 3 warpgroups
constexpr int kKProducerWarp = 8;
constexpr int kMmaWarp0 = 9;
constexpr int kVProducerWarp = 10;
constexpr int kMmaWarp1 = 11;
// setmaxnreg: the kernel launches with 168 registers/thread (65536 / 384); the two softmax warpgroups grow to
// 208 (a full S row lives in registers), the producer/MMA warpgroup shrinks to 88.  The registers the 128
// threads give up must cover what the 256 softmax threads take, or setmaxnreg.inc never returns.
#ifndef DSA_REGS_SOFTMAX
#define DSA_REGS_SOFTMAX 208
#define DSA_REGS_OTHER 88
#endif
constexpr int kRegsLaunch = 168;
constexpr int kRegsSoftmax = DSA_REGS_SOFTMAX;
constexpr int kRegsOther = DSA_REGS_OTHER;
static_assert((kRegsLaunch - kRegsOther) * 128 >= (kRegsSoftmax - kRegsLaunch) * 256, "setmaxnreg pool imbalance");
constexpr int kTmemCols = 512;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
// lazy rescale: O and l are only rescaled when the row max grew by more than 2^8 (log2 domain).
constexpr float kRescaleThreshold = 8.0f;
// Early issue of the second half of S_x(j+1) (keys [BC/2, BC), columns P_x(j) does not use) as soon as S_x(j) is in
// registers.  Measured slower on B200 (dense cfg1 11.3 ms against 10.1 ms): with A = Q_x read from shared memory every
// N = BC/2 instruction still reads the whole 4 KB A tile, so two half-width Q K^T cost ~1.5x one full-width one.  Off.
#ifndef DSA_EARLY_B
#define DSA_EARLY_B 0
#endif
#ifndef DSA_F32X2
#define DSA_F32X2 1
#endif
#ifndef DSA_EXP
#define DSA_EXP 0   // timing experiments only (results are wrong unless nothing is skipped)
#endif
#ifndef DSA_EXP_LOCK
#define DSA_EXP_LOCK 0
#endif
// number of tcgen05.mma issuer warps (1: warp 9 drives both slots; 2: one warp per slot)
#ifndef DSA_GATE
#define DSA_GATE 1
#endif
#ifndef DSA_ISSUERS_DENSE
#define DSA_ISSUERS_DENSE 1
#endif
#ifndef DSA_ISSUERS_SPARSE
#define DSA_ISSUERS_SPARSE 2
#endif

struct FwdArgs {
    __nv_bfloat16* out;          // [BH, N, D]
    float* lse;                  // [BH, N] or null
    unsigned long long* stats;   // [BH, 2] or null (pre-zeroed)
    uint8_t* skip_mask;          // [BH, T_r, T_c_dec] or null
    float* margin;               // [BH, T_r, T_c_dec] or null
    const float* lse_in;         // MASS mode: dense lse [BH, N], natural log
    float* mass_out;             // MASS mode: [BH, T_r, T_c] fp32, pre-zeroed: sum over the tile of e^(S - lse)
    const uint8_t* mask_in;      // MASK mode: [BH, T_r, T_c] bytes, non-zero = skip (tile 0 is kept regardless)
    int N;
    int T_r;                     // decision tiles along queries
    int T_c;                     // K tiles of BC keys (MMA tiles)
    int T_c_dec;                 // decision tiles along keys: ceil(N / tile_k), = T_c unless tile_k < BC
    int n_mma_tiles;             // ceil(N / 128)
    int mode;
    float scale_log2;            // softmax_scale * log2(e)
    float lambda_log2;           // lambda * log2(e)
#ifdef DSA_PROF
    unsigned long long* prof;    // [n_cta][32] cycle counters (profiling builds only)
#endif
};

template <int D, int BC, int NK, int NV>
struct SmemLayout {
    static constexpr int kQSlotBytes = 128 * D * 2;
    static constexpr int kSubQBytes = 128 * 128;        // one 64-column (128 B) sub-tile of Q
    static constexpr int kKVStageBytes = BC * D * 2;
    static constexpr int kSubKVBytes = BC * 128;        // one 64-column sub-tile of K or V
    static constexpr int kQOff = 0;
    static constexpr int kKOff = 2 * kQSlotBytes;
    static constexpr int kVOff = kKOff + NK * kKVStageBytes;
    static constexpr int kBarOff = kVOff + NV * kKVStageBytes;
    // barriers (8 B each): q_full[2] k_full[NK] k_empty[NK] v_full[NV] v_empty[NV]
    //                      s_full[2] p_half[2] p_ready[2] o_full[2] s_read[2] dec[2][4]
    static constexpr int kNumBars = 2 + 2 * NK + 2 * NV + 8 + 2 + 8;
    static constexpr int kMiscOff = kBarOff + 8 * kNumBars;
    // misc: tmem_ptr (4) | pad (12) | votes[2][4][4] (128) | wmax[2][4][4] (128) | in_exp[2][4] (32) | prog[2] (16) | pvmask[2][4] (32)
    static constexpr int kVotesOff = kMiscOff + 16;
    static constexpr int kLockOff = kVotesOff + 256;
    static constexpr int kProgOff = kLockOff + 32;
    static constexpr int kPvMaskOff = kProgOff + 16;       // pvmask[2][4]: kept sub-tiles of tile j (SUB > 1), ring like votes
    static constexpr int kPreOff = kPvMaskOff + 32;        // pre[2][4][4]: per-warp votes on sub-tiles (SUB > 1): buffers 0, 1
                                                           // preliminary round of tile j (by parity), 2, 3 later rounds
    static constexpr int kMiscBytes = 16 + 128 + 128 + 32 + 16 + 32 + 128;
    static constexpr int kTotal = kMiscOff + kMiscBytes;
    static constexpr int kDynamicBytes = kTotal + 1024;  // slack for the 1024-B alignment of the swizzled tiles
    static_assert(kDynamicBytes <= 232448, "exceeds the 227 KB of shared memory a CTA may use");
};

// kSparse = false compiles the DENSE mode only (no predicate, no vote, V always fetched);
// kDebug adds the optional skip_mask_out / margin_out parity outputs.
// SUB == 0: the block-mass kernel of sparse_attn_block_mass (its own instantiation, so that the forward kernels carry none
// of its code: a run-time branch for it inside the sparse kernels cost them 7-9 %).
// SUB > 1 (sparse modes, G = 1): the decision tile is BR x (BC / SUB) keys -- SUB decisions per MMA tile, taken in
// ascending key order with the statistics updated after every retained one (block size 32).
template <int D, int BC, int G, int NK, int NV, bool kSparse, bool kDebug, int SUB = 1>
__global__ void __launch_bounds__(kNumThreads, 1)
sparse_attn_fwd_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                       const __grid_constant__ CUtensorMap tm_v, const FwdArgs a) {
    using L = SmemLayout<D, BC, NK, NV>;
    static_assert(D == 64 || D == 128, "head dim");
    static_assert(BC == 64 || BC == 128, "key tile");
    static_assert(2 * BC + 2 * D <= kTmemCols, "TMEM budget");
    constexpr bool kMass = SUB == 0;
    constexpr int kSubN = SUB > 0 ? SUB : 1;
    static_assert(SUB == 1 || (kMass && kSparse && !kDebug) ||
                  (kSparse && G == 1 && (SUB == 2 || SUB == 4) && (BC / kSubN) % 32 == 0), "sub-tile decisions / mass kernel");
    constexpr int BR = 128 / G;
    constexpr int kSubD = D / 64;
    constexpr uint32_t kIdescQK = umma_idesc_bf16(128, BC, 0);   // S = Q K^T: A, B both K-major
    constexpr uint32_t kIdescQKh = umma_idesc_bf16(128, BC / 2, 0);   // one half of the keys of a tile
    constexpr uint32_t kIdescPV = umma_idesc_bf16(128, D, 1);    // O += P V: B = V is MN-major (d contiguous)

    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t sbase = (raw + 1023u) & ~1023u;
    uint8_t* smem = smem_raw + (sbase - raw);

    const uint32_t q_smem = sbase + L::kQOff;
    const uint32_t k_smem = sbase + L::kKOff;
    const uint32_t v_smem = sbase + L::kVOff;
    const uint32_t bar0 = sbase + L::kBarOff;
    auto q_full = [&](int x) { return bar0 + 8u * x; };
    auto k_full = [&](int s) { return bar0 + 8u * (2 + s); };
    auto k_empty = [&](int s) { return bar0 + 8u * (2 + NK + s); };
    auto v_full = [&](int s) { return bar0 + 8u * (2 + 2 * NK + s); };
    auto v_empty = [&](int s) { return bar0 + 8u * (2 + 2 * NK + NV + s); };
    constexpr int kB = 2 + 2 * NK + 2 * NV;
    auto s_full = [&](int x) { return bar0 + 8u * (kB + x); };        // S_X(j) complete in TMEM
    auto p_half = [&](int x) { return bar0 + 8u * (kB + 2 + x); };    // first half of P_X written (kept tiles only)
    auto p_ready = [&](int x) { return bar0 + 8u * (kB + 4 + x); };   // all of P_X written (kept tiles only)
    auto o_full = [&](int x) { return bar0 + 8u * (kB + 6 + x); };    // last P V of slot X complete
    auto s_read = [&](int x) { return bar0 + 8u * (kB + 8 + x); };    // the 4 warps of slot X hold S_X(j) in registers
    // the 4 warps of slot X have voted on tile j.  A ring of 4 barriers (and 4 vote words per warp), indexed by
    // j & 3: the votes are read by the slot's MMA warp, by the V warp and by the slot's own all-skip warps.  Slot x
    // can only vote on tile j + 3 after its MMA warp has finished tile j + 1, which waits for v_full of tile j + 1,
    // which the V warp completes only after it has read every vote on tile j: a ring of 4 can never be lapped.
    auto dec = [&](int x, int q) { return bar0 + 8u * (kB + 10 + 4 * x + q); };
    volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(smem + L::kMiscOff);
    volatile int* votes = reinterpret_cast<volatile int*>(smem + L::kVotesOff);                  // [2][4][4]
    volatile float* wmax = reinterpret_cast<volatile float*>(smem + L::kVotesOff + 128);         // [2][4][4]

    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);   // warp-uniform: role and slot indices live in uniform registers
    const int lane = threadIdx.x & 31;
    const int bh = blockIdx.y;
    const int tile0 = blockIdx.x * 2;
    const bool active1 = (tile0 + 1) < a.n_mma_tiles;
    const int nX = active1 ? 2 : 1;
    const int T_c = a.T_c;

    // ------------------------------------------------------------------ setup
    if (warp == kKProducerWarp && lane == 0) {
        prefetch_tmap(&tm_q);
        prefetch_tmap(&tm_k);
        prefetch_tmap(&tm_v);
        for (int x = 0; x < 2; ++x) {
            mbar_init(q_full(x), 1);
            mbar_init(s_full(x), 1);
            mbar_init(p_half(x), 128);
            mbar_init(p_ready(x), 128);
            mbar_init(o_full(x), 1);
            for (int q = 0; q < 4; ++q) mbar_init(dec(x, q), 4);
            mbar_init(s_read(x), 4);
        }
        // a K stage is released by one softmax lane per active slot (when S_x of that tile is complete),
        // a V slot by the MMA warp of every active slot (after its P V, or at once if it skipped the tile)
        for (int s = 0; s < NK; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), nX); }
        for (int s = 0; s < NV; ++s) { mbar_init(v_full(s), 1); mbar_init(v_empty(s), nX); }
        for (int i = 0; i < 32; ++i) votes[i] = -1;
        for (int i = 0; i < 12; ++i) reinterpret_cast<volatile int*>(smem + L::kLockOff)[i] = 0;  // in_exp, prog
        fence_mbar_init();
    }
    if (warp == kMmaWarp0) {
        tmem_alloc(smem_u32(const_cast<uint32_t*>(tmem_ptr)), kTmemCols);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    if (warp >= 8) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsOther));
        // Producer / MMA warps: the whole warp runs each loop (warp-uniform control flow, every lane waits on
        // the mbarriers) and one elected lane issues, so that descriptors and addresses stay in uniform registers.
        if (warp == kKProducerWarp) {
            // ========================================================== Q and K producer (a1)
            if (elect_one_sync()) {
                for (int x = 0; x < nX; ++x) {
                    mbar_arrive_expect_tx(q_full(x), L::kQSlotBytes);
                    for (int h = 0; h < kSubD; ++h)
                        tma_load_3d(q_smem + x * L::kQSlotBytes + h * L::kSubQBytes, &tm_q, h * 64,
                                    (tile0 + x) * 128, bh, q_full(x));
                }
            }
            __syncwarp();
            int stage = 0;
            uint32_t phase = 0;
            for (int j = 0; j < T_c; ++j) {
                if (j >= NK) mbar_wait(k_empty(stage), phase ^ 1u);
                if (elect_one_sync()) {
                    mbar_arrive_expect_tx(k_full(stage), L::kKVStageBytes);
                    for (int h = 0; h < kSubD; ++h)
                        tma_load_3d(k_smem + stage * L::kKVStageBytes + h * L::kSubKVBytes, &tm_k, h * 64, j * BC, bh,
                                    k_full(stage));
                }
                __syncwarp();
                if (++stage == NK) { stage = 0; phase ^= 1u; }
            }
        } else if (warp == kVProducerWarp) {
            // ========================================================== V producer (a1)
            // V_j lives in ring slot j % NV, and v_full / v_empty of that slot complete exactly one phase per tile
            // mapped to it, whether V_j was fetched or not, so every waiter's phase parity is a function of j alone.
            auto wait_slot_free = [&](int j) {               // tile j - NV has been released by every active slot
                if (j >= NV) mbar_wait(v_empty(j % NV), static_cast<uint32_t>((j / NV) - 1) & 1u);
            };
            auto load_v = [&](int j) {
                const int slot = j % NV;
                wait_slot_free(j);
                if (elect_one_sync()) {
                    mbar_arrive_expect_tx(v_full(slot), L::kKVStageBytes);
                    for (int h = 0; h < kSubD; ++h)
                        tma_load_3d(v_smem + slot * L::kKVStageBytes + h * L::kSubKVBytes, &tm_v, h * 64, j * BC, bh,
                                    v_full(slot));
                }
                __syncwarp();
            };
            if (!kSparse || (DSA_EXP & 4)) {
                for (int j = 0; j < T_c; ++j) load_v(j);
            } else {
                // Sparse modes: V_j is needed iff some slot keeps tile j.  This warp reads the votes of both slots
                // (barrier dec), fetches V_j if it is needed and not yet there, and after a kept tile fetches V_{j+1}
                // ahead of its votes (decisions are strongly correlated along j); a wasted prefetch costs L2 traffic
                // only.  A tile nobody keeps completes its v_full phase with a plain arrive.
                load_v(0);                                   // tile 0 is always kept
                bool have = true;                            // is V_j already in (or on its way to) its slot?
                for (int j = 0; j < T_c; ++j) {
                    const int q = j & 3;
                    const int tag_keep = (j << 2) | 2;
                    const bool has_next = (j + 1) < T_c;
                    bool have_next = false;
                    bool keep = false;
                    for (int x = 0; x < nX; ++x) {           // act on the first keep vote, do not wait for both slots
                        mbar_wait(dec(x, q), (j >> 2) & 1);
                        const int4 vt = lds128_volatile(sbase + L::kVotesOff + (x * 4 + q) * 16);
                        keep |= (vt.x == tag_keep) | (vt.y == tag_keep) | (vt.z == tag_keep) | (vt.w == tag_keep);
                        if (keep) {
                            if (!have) { load_v(j); have = true; }
                            if (has_next && !have_next) { load_v(j + 1); have_next = true; }
                        }
                    }
                    if (!have) {                             // nobody keeps tile j: complete its phase without a load
                        wait_slot_free(j);
                        if (lane == 0) mbar_arrive(v_full(j % NV));
                        __syncwarp();
                    }
                    have = have_next;
                }
            }
        } else if (warp == kMmaWarp0 || warp == kMmaWarp1) {
            // ========================================================== MMA issuer(s) (a2, a6)
            // kIssuers == 2: warp 9 drives slot 0 and warp 11 slot 1.  kIssuers == 1: warp 9 drives both slots in turn
            // (warp 11 idles), which forces the two slots into anti-phase -- the best schedule when every tile is kept.
            constexpr int kIssuers = kSparse ? DSA_ISSUERS_SPARSE : DSA_ISSUERS_DENSE;
            constexpr bool kGate = kIssuers == 2 && DSA_GATE;
            constexpr bool kEarlyB = DSA_EARLY_B;
            const int x_lo = (kIssuers == 2 && warp == kMmaWarp1) ? 1 : 0;
            const int x_hi = (kIssuers == 2) ? x_lo + 1 : nX;        // this warp drives slots [x_lo, x_hi)
            if ((kIssuers == 2 || warp == kMmaWarp0) && x_lo < nX) {
            // S_x = Q_x K^T for the keys of half h of the tile (h = 0: keys [0, BC/2) -> columns [0, BC/2) of S_x,
            // h = 1: the other half; h = 2: the whole tile in one N = BC instruction per k step)
            auto issue_qk = [&](int x, uint32_t kaddr, int h = 2) {
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t off = (kk >> 2) * L::kSubQBytes + (kk & 3) * 32;
                    const uint32_t koff = (kk >> 2) * L::kSubKVBytes + (kk & 3) * 32 + (h == 1 ? (BC / 2) * 128 : 0);
                    umma_ss(tmem_base + x * BC + (h == 1 ? BC / 2 : 0),
                            umma_smem_desc_sw128(q_smem + x * L::kQSlotBytes + off, 16, 1024),
                            umma_smem_desc_sw128(kaddr + koff, 16, 1024), h == 2 ? kIdescQK : kIdescQKh, kk > 0);
                }
            };
            // half 0 / 1: keys [0, BC/2) / [BC/2, BC); mask (SUB > 1): bit s set = decision sub-tile s was kept
            auto issue_pv = [&](int x, uint32_t vaddr, bool acc, int half, uint32_t mask = 0xffu) {
#pragma unroll
                for (int kk = half * (BC / 32); kk < (half + 1) * (BC / 32); ++kk) {
                    if (SUB > 1 && !((mask >> (kk / (BC / 16 / kSubN))) & 1u)) continue;   // P of a skipped sub-tile is never read
                    // 16 keys = 16 rows of 128 B; d sub-tiles (64 columns) are L::kSubKVBytes apart (LBO)
                    umma_ts(tmem_base + 2 * BC + x * D, tmem_base + x * BC + kk * 8,
                            umma_smem_desc_sw128(vaddr + kk * 2048, L::kSubKVBytes, 1024), kIdescPV, acc || kk > 0);
                }
            };
            int kstage = 0;
            uint32_t kphase = 0;
            for (int x = x_lo; x < x_hi; ++x) mbar_wait(q_full(x), 0);
            mbar_wait(k_full(0), 0);
            tc_fence_after();
            if (elect_one_sync()) {
                for (int x = x_lo; x < x_hi; ++x) {
                    issue_qk(x, k_smem);
                    umma_commit(s_full(x));
                }
            }
            __syncwarp();
            if (++kstage == NK) { kstage = 0; kphase ^= 1u; }
            uint32_t ppar[2] = {0u, 0u};                 // parity of p_half / p_ready: they advance on kept tiles only
            bool prev_skip[2] = {false, false};          // did slot x skip tile j-1?
            // Sparse modes, speculation: inside a run of skipped tiles the next S_x(j+1) = Q_x K_{j+1}^T is issued as
            // soon as the softmax warps hold S_x(j) in registers (barrier s_read), without waiting for their vote:
            // the vote is then off the critical chain.  If tile j turns out to be kept, the softmax warps let the
            // speculative MMA finish before they write P_x over it, and S_x(j+1) is issued again after P_x V_j.
            // Scheduling only: no decision depends on it.
            for (int j = 0; j < T_c; ++j) {
                const bool has_next = (j + 1) < T_c;
                const int vslot = j % NV;
                const uint32_t vph = static_cast<uint32_t>(j / NV) & 1u;
                const uint32_t vaddr = v_smem + vslot * L::kKVStageBytes;
                const uint32_t kaddr = k_smem + kstage * L::kKVStageBytes;
                if (has_next) { mbar_wait(k_full(kstage), kphase); tc_fence_after(); }   // K_{j+1} has landed
#pragma unroll
                for (int x = 0; x < 2; ++x) {
                    if (x < x_lo || x >= x_hi) continue;
                    // As soon as the softmax warps hold S_x(j) in registers (barrier s_read), the second half of
                    // S_x(j+1) is issued: its columns are not needed for P_x(j), which occupies the first BC/2 columns
                    // only, so this half of the next Q K^T is off the chain P ready -> P V -> Q K^T -> S ready.
                    // In a run of skipped tiles the first half follows at once (speculation, see above).
                    const bool spec = kSparse && prev_skip[x] && has_next;
                    if (has_next && (kEarlyB || spec)) {
                        mbar_wait(s_read(x), j & 1);
                        TRACE(12)
                        tc_fence_after();
                        if (elect_one_sync()) {
                            if (kEarlyB) issue_qk(x, kaddr, 1);
                            if (spec) {
                                issue_qk(x, kaddr, kEarlyB ? 0 : 2);
                                umma_commit(s_full(x));
                            }
                        }
                        __syncwarp();
                        TRACE(13)
                    }
                    bool keep = true;
                    if (kSparse && !(DSA_EXP & 2)) {
                        TRACE(0)
                        const int q = j & 3;
                        mbar_wait(dec(x, q), (j >> 2) & 1);  // all 4 warps of slot x have voted on tile j
                        tc_fence_after();                    // (their votes follow their tcgen05.ld of S_x(j))
                        TRACE(1)
                        const int tag_keep = (j << 2) | 2;
                        const int4 vt = lds128_volatile(sbase + L::kVotesOff + (x * 4 + q) * 16);
                        keep = (vt.x == tag_keep) | (vt.y == tag_keep) | (vt.z == tag_keep) | (vt.w == tag_keep);
                        prev_skip[x] = !keep;
                    }
                    if (kGate && nX == 2 && keep) {
                        // two issuers: the P V phases of two slots that both keep their tiles still take turns in the
                        // order (0, j), (1, j), (0, j+1), ... as they would with one issuer, which holds the slots in
                        // anti-phase (softmax of one under the MMAs of the other); a slot that skips never waits, and
                        // the speculative issues above run side by side.  Scheduling only.
                        const int need = (x == 0) ? j : j + 1;
                        while (static_cast<int>(ld_shared_u32(sbase + L::kProgOff + 4 * (1 - x))) < need) { }
                    }
                    if (keep) {
                        mbar_wait(p_half(x), ppar[x]);
                        mbar_wait(v_full(vslot), vph);       // V_j has landed (sparse modes: fetched by the V warp
                        tc_fence_after();                    // once some slot voted to keep tile j, or prefetched)
                        uint32_t pvmask = 0xffu;
                        if (SUB > 1) pvmask = ld_shared_u32(sbase + L::kPvMaskOff + (x * 4 + (j & 3)) * 4);
                        if (elect_one_sync()) issue_pv(x, vaddr, j > 0, 0, pvmask);
                        __syncwarp();
                        mbar_wait(p_ready(x), ppar[x]);
                        tc_fence_after();
                        ppar[x] ^= 1u;
                        uint32_t pvmask2 = 0xffu;            // the mask is complete once all of P_x has been handed over
                        if (SUB > 1) pvmask2 = ld_shared_u32(sbase + L::kPvMaskOff + (x * 4 + (j & 3)) * 4);
                        TRACE(2)
                        if (elect_one_sync()) {
                            issue_pv(x, vaddr, true, 1, pvmask2);
                            umma_commit(v_empty(vslot));     // this slot's P_x V_j has read V_j
                            if (has_next) {
                                issue_qk(x, kaddr, kEarlyB ? 0 : 2);   // (again, if a speculative one was overwritten by P_x)
                                umma_commit(s_full(x));
                            } else {
                                umma_commit(o_full(x));
                            }
                        }
                        __syncwarp();
                    } else {
                        TRACE(2)
                        if (!spec) {
                            if (elect_one_sync()) {
                                if (has_next) {
                                    issue_qk(x, kaddr, kEarlyB ? 0 : 2);
                                    umma_commit(s_full(x));
                                } else {
                                    umma_commit(o_full(x));
                                }
                            }
                            __syncwarp();
                        }
                        // the V warp has dealt with tile j (and a prefetched but unused V_j has landed): release the slot
                        mbar_wait(v_full(vslot), vph);
                        if (lane == 0) mbar_arrive(v_empty(vslot));
                        __syncwarp();
                    }
                    if (kGate && nX == 2 && lane == 0) st_shared_u32(sbase + L::kProgOff + 4 * x, static_cast<uint32_t>(j + 1));
                    TRACE(3)
                }
                if (has_next && ++kstage == NK) { kstage = 0; kphase ^= 1u; }
            }
            }
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsSoftmax));
        if (warp < 4 * nX) {
        // ============================================================== softmax warpgroups (a3-a5, a7-a9)
        const int x = warp >> 2;
        const int w = warp & 3;
        const int r = threadIdx.x & 127;
        const uint32_t lane_base = static_cast<uint32_t>(w * 32) << 16;
        const uint32_t tS = tmem_base + lane_base + x * BC;
        const uint32_t tO = tmem_base + lane_base + 2 * BC + x * D;
        const int mma_tile = tile0 + x;
        const int grow = mma_tile * 128 + r;
        const bool row_valid = grow < a.N;
        const int grp = (G == 2) ? (w >> 1) : 0;
        const int dtile = mma_tile * G + grp;
        const bool grp_valid = dtile < a.T_r;
        const bool grp_leader = (r % BR) == 0;
        const size_t tile_row = (static_cast<size_t>(bh) * a.T_r + dtile) * static_cast<size_t>(a.T_c_dec);
        const int mode = a.mode;
        const float scale_log2 = a.scale_log2;
        const float lambda_log2 = a.lambda_log2;
        const bool want_margin = kDebug && a.margin != nullptr;

        constexpr bool kUseExpLock = DSA_EXP_LOCK == 2 || (DSA_EXP_LOCK == 1 && (kSparse ? DSA_ISSUERS_SPARSE : DSA_ISSUERS_DENSE) == 2);
        // MASS mode: -lse_r in log2 units (+... rows beyond N contribute nothing)
        float neg_lse2 = -INFINITY;
        if (kMass && row_valid) neg_lse2 = -a.lse_in[static_cast<size_t>(bh) * a.N + grow] * kLog2e;
        float m_used = -INFINITY;   // stabiliser actually subtracted (log2 domain, may lag the true max)
        float m_true = -INFINITY;   // running max over retained tiles (log2 domain) -- FIXED mode reference
        float l = 0.f;              // sum over retained tiles of 2^(s - m_used)
        float lse2 = -INFINITY;     // m_used + log2(l): LSE over retained tiles, log2 domain (Eq. 6) -- DYNAMIC reference
        int n_exec = 0, n_skip = 0;
        uint32_t sfpar = 0;         // parity of s_full(x): one phase per S_x issued (two for a tile re-issued after a
                                    // mis-speculated skip)
        bool prev_skip = false;     // did this slot skip tile j-1?
        PROF_DECL(8)

        for (int j = 0; j < T_c; ++j) {
            PROF_TICK(0)
            if (w == 0) { TRACE(4) }
            // MASK mode: this tile's byte is fetched before the wait for S_x(j), which hides the global-memory latency
            bool mask_skip = false;
            if (kSparse && mode == kModeMask) mask_skip = (j > 0) && (!grp_valid || __ldg(a.mask_in + tile_row + j) != 0);
            mbar_wait(s_full(x), sfpar);
            sfpar ^= 1u;
            tc_fence_after();
            // S_x(j) is complete, so this slot's Q K^T has read K_j for the last time (a mis-speculated S_x(j) was
            // consumed, and issued again, during tile j-1): release this slot's hold on the K stage
            if (w == 0 && lane == 0) mbar_arrive(k_empty(j % NK));
            if (w == 0) { TRACE(5) }
            PROF_TICK(1)
            uint32_t su[BC / 32][32];                         // this thread's row of S_ij (fp32 bits)
#pragma unroll
            for (int c = 0; c < BC / 32; ++c) tmem_ld_x32(tS + c * 32, su[c]);
            tmem_wait_ld();
            // inside a run of skipped tiles the MMA warp issues S_x(j+1) as soon as S_x(j) has left TMEM
            const bool spec = kSparse && prev_skip && (j + 1) < T_c;
            if (kSparse || DSA_EARLY_B) {                    // S_x(j) has left TMEM
                tc_fence_before();
                if (lane == 0) mbar_arrive(s_read(x));
            }
            if (w == 0) { TRACE(6) }
            PROF_TICK(2)
#define S_AT(c) __uint_as_float(su[(c) >> 5][(c) & 31])
            const int valid_cols = a.N - j * BC;             // ragged last K tile: columns beyond N are -inf
            if (valid_cols < BC) {
#pragma unroll
                for (int c = 0; c < BC; ++c)
                    if (c >= valid_cols) su[c >> 5][c & 31] = 0xff800000u;
            }
            if constexpr (kMass) {
                // Block mass of the dense attention probabilities: sum over the rows of this warp and the columns of the
                // tile of e^(S_rc - lse_r) (the quantity Top-K / Top-P block selection ranks).  No P, no
                // P V: the tile is voted "skipped", so the issuer streams Q K^T only.
                float acc0 = 0.f, acc1 = 0.f;
#pragma unroll
                for (int c = 0; c < BC; c += 2) {
                    acc0 += fast_exp2(fmaf(S_AT(c), scale_log2, neg_lse2));
                    acc1 += fast_exp2(fmaf(S_AT(c + 1), scale_log2, neg_lse2));
                }
                float acc = row_valid ? acc0 + acc1 : 0.f;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
                if (lane == 0 && grp_valid) atomicAdd(a.mass_out + tile_row + j, acc);
                tc_fence_before();
                if (lane == 0) {
                    votes[(x * 4 + (j & 3)) * 4 + w] = (j << 2) | 1;
                    mbar_arrive(dec(x, j & 3));
                }
                __syncwarp();
                prev_skip = true;
                continue;
            }
            float mx0 = S_AT(0), mx1 = S_AT(1), mx2 = S_AT(2), mx3 = S_AT(3);   // 4 independent 3-input max chains
#pragma unroll
            for (int c = 4; c + 8 <= BC; c += 8) {
                mx0 = fmax3(mx0, S_AT(c), S_AT(c + 1));
                mx1 = fmax3(mx1, S_AT(c + 2), S_AT(c + 3));
                mx2 = fmax3(mx2, S_AT(c + 4), S_AT(c + 5));
                mx3 = fmax3(mx3, S_AT(c + 6), S_AT(c + 7));
            }
            mx0 = fmax3(mx0, S_AT(BC - 4), S_AT(BC - 3));
            mx1 = fmax3(mx1, S_AT(BC - 2), S_AT(BC - 1));
            const float mhat2 = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * scale_log2;   // tile-local row max (a3)
            if (w == 0) { TRACE(7) }
            PROF_TICK(3)

            if constexpr (SUB > 1) {
                // ============ decision tiles of BC / SUB keys: SUB decisions per MMA tile, in key order
                constexpr int W = BC / SUB;                  // keys per decision tile (32 or 64)
                const int q = j & 3;
                // the stabiliser m_used follows the max of the WHOLE MMA tile (it only has to bound the exponents; a
                // sub-tile with a large max is never skipped), so it is fixed before any P of this tile is written
                if (j == 0) {
                    m_used = mhat2;
                } else {
                    const bool need = mhat2 > m_used + kRescaleThreshold;
                    if (__any_sync(0xffffffffu, need)) {
                        const float alpha = need ? fast_exp2(m_used - mhat2) : 1.f;
                        if (need) m_used = mhat2;
                        l *= alpha;                          // (m_used + log2 l, hence lse2, is unchanged)
#pragma unroll
                        for (int c = 0; c < D / 32; ++c) {   // O_r *= alpha (PV of tile j-1 has completed: s_full(j))
                            uint32_t o[32];
                            tmem_ld_x32(tO + c * 32, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                            tmem_st_x32(tO + c * 32, o);
                        }
                    }
                }
                const float neg_m = -m_used;
                const uint64_t scale2 = pack_f32x2(scale_log2, scale_log2);
                const uint64_t negm2 = pack_f32x2(neg_m, neg_m);
                // Row maxima of the SUB decision tiles (a3), then a PRELIMINARY test of all of them against the
                // statistics as they stand before this MMA tile.  Within the tile the reference (LSE, or the running
                // max) can only grow, so t can only shrink: a sub-tile skipped by the preliminary test is skipped by
                // the sequential rule too.  One vote round settles every skipped sub-tile (all of them in a run of
                // skipped tiles); only sub-tiles that pass it AND follow a retained one are tested again.
                float msub[SUB];
#pragma unroll
                for (int s = 0; s < SUB; ++s) {
                    float ma = S_AT(s * W), mb = S_AT(s * W + 1), mc = S_AT(s * W + 2), md = S_AT(s * W + 3);
#pragma unroll
                    for (int c = 4; c + 8 <= W; c += 8) {    // 4 independent 3-input max chains
                        ma = fmax3(ma, S_AT(s * W + c), S_AT(s * W + c + 1));
                        mb = fmax3(mb, S_AT(s * W + c + 2), S_AT(s * W + c + 3));
                        mc = fmax3(mc, S_AT(s * W + c + 4), S_AT(s * W + c + 5));
                        md = fmax3(md, S_AT(s * W + c + 6), S_AT(s * W + c + 7));
                    }
                    ma = fmax3(ma, S_AT(s * W + W - 4), S_AT(s * W + W - 3));
                    mb = fmax3(mb, S_AT(s * W + W - 2), S_AT(s * W + W - 1));
                    msub[s] = fmaxf(fmaxf(ma, mb), fmaxf(mc, md)) * scale_log2;
                }
                uint32_t cand = (1u << SUB) - 1u;            // bit s: sub-tile s passed the preliminary test; bit SUB+s: kept for certain
                if (!kDebug) {                               // (debug builds test every sub-tile in sequence: margins)
                    const float ref0 = (mode == kModeDynamic) ? lse2 : m_true;
                    // Upper bound of how far the reference of this row can grow inside the tile, whatever is retained:
                    // LSE' <= log2(2^LSE + BC * 2^mhat) (DYNAMIC), m' <= max(m, mhat) (FIXED).  A row whose t stays
                    // >= lambda even against that bound keeps its sub-tile for certain, with no second vote (bits
                    // SUB..2 SUB-1).  1e-3 covers the rounding of the approximate ex2 / lg2 in the running statistics.
                    const float grow = ((mode == kModeDynamic) ? fast_log2(1.f + static_cast<float>(BC) * fast_exp2(mhat2 - ref0))
                                                               : fmaxf(0.f, mhat2 - ref0)) + 1e-3f;
                    uint32_t wc = 0u;
#pragma unroll
                    for (int s = 0; s < SUB; ++s) {
                        const bool rs = (j * SUB + s > 0) && (!row_valid || (msub[s] - ref0 < lambda_log2));
                        if (!__all_sync(0xffffffffu, rs)) wc |= 1u << s;
                        const bool sure = row_valid && (msub[s] - ref0 - grow >= lambda_log2);
                        if (__any_sync(0xffffffffu, sure)) wc |= 1u << (SUB + s);
                    }
                    volatile uint32_t* pre = reinterpret_cast<volatile uint32_t*>(smem + L::kPreOff) + (x * 4 + (j & 1)) * 4;
                    if (lane == 0) pre[w] = wc;
                    named_bar_sync(1 + x, 128);
                    cand = pre[0] | pre[1] | pre[2] | pre[3];
                }
                uint32_t kept = 0u;                          // bit s: decision sub-tile s retained
                bool half_sent = false;
                // Row sums of retained sub-tiles are folded into l (and LSE) lazily: only a decision that is still open
                // needs the new LSE (Eq. 6); between sub-tiles that are settled the ex2 streams run back to back.
                uint64_t acc2 = pack_f32x2(0.f, 0.f);
                bool dirty = false;
                auto fold = [&]() {
                    if (dirty) {
                        float r0, r1;
                        unpack_f32x2(acc2, r0, r1);
                        l += r0 + r1;
                        if (mode == kModeDynamic) lse2 = m_used + fast_log2(l);
                        acc2 = pack_f32x2(0.f, 0.f);
                        dirty = false;
                    }
                };
#pragma unroll
                for (int s = 0; s < SUB; ++s) {
                    const int jj = j * SUB + s;              // decision tile index along the keys
                    if (jj >= a.T_c_dec) break;              // beyond the last key (ragged tail): no such tile
                    const float ms = msub[s];
                    const bool open = ((cand >> s) & 1u) && (kDebug || (kept != 0u && !((cand >> (SUB + s)) & 1u)));
                    if (open) fold();                        // this decision is taken with the current statistics
                    const float ref = (mode == kModeDynamic) ? lse2 : m_true;
                    const float t2 = ms - ref;               // Eq. 5, log2 units (+inf before the first retained tile)
                    const bool row_skip = (jj > 0) && (!row_valid || (t2 < lambda_log2));
                    uint64_t rs2 = pack_f32x2(0.f, 0.f);     // row sum of this sub-tile, two packed chains
                    auto exp_sub = [&]() {                   // a5 for this sub-tile: P columns and row sum
#pragma unroll
                        for (int c = s * (W / 32); c < (s + 1) * (W / 32); ++c) {
                            uint32_t pk[16];
#pragma unroll
                            for (int i = 0; i < 16; ++i) {
                                float x0, x1;
                                unpack_f32x2(fma_f32x2(pack_f32x2(__uint_as_float(su[c][2 * i]), __uint_as_float(su[c][2 * i + 1])),
                                                       scale2, negm2), x0, x1);
                                const float p0 = fast_exp2(x0);
                                const float p1 = fast_exp2(x1);
                                rs2 = add_f32x2(rs2, pack_f32x2(p0, p1));
                                pk[i] = pack_bf16x2(p0, p1);
                            }
                            tmem_st_x16(tS + c * 16, pk);
                        }
                    };
                    bool skip_s, did_exp = false;
                    if (!((cand >> s) & 1u)) {
                        skip_s = true;                       // settled by the preliminary round
                    } else if (!kDebug && (kept == 0u || ((cand >> (SUB + s)) & 1u))) {
                        skip_s = false;                      // statistics unchanged since that round, or kept for certain
                    } else if (kept != 0u) {
                        // A sub-tile that follows a retained one is exponentiated BEFORE its vote is settled: the
                        // all-rows vote (shared-memory words + one barrier) then completes in the shadow of the ex2
                        // work instead of holding it up.  If the vote says skip, the P columns just written are never
                        // read (mask bit clear) and the row sum is dropped.
                        exp_sub();
                        did_exp = true;
                        const bool wv = __all_sync(0xffffffffu, row_skip);
                        volatile uint32_t* sv = reinterpret_cast<volatile uint32_t*>(smem + L::kPreOff) + (x * 4 + 2 + (s & 1)) * 4;
                        if (lane == 0) sv[w] = wv ? 1u : 0u;
                        named_bar_sync(1 + x, 128);
                        skip_s = (sv[0] & sv[1] & sv[2] & sv[3]) != 0u;   // all 128 rows of the Q tile (R1)
                    } else {
                        skip_s = named_bar_red_and(1 + x, 128, row_skip);
                    }
                    if (kDebug) {
                        float gm = INFINITY;
                        if (want_margin) {
                            float tm = row_valid ? t2 : -INFINITY;
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) tm = fmaxf(tm, __shfl_xor_sync(0xffffffffu, tm, o));
                            if (lane == 0) wmax[(x * 4 + q) * 4 + w] = tm;
                            named_bar_sync(1 + x, 128);
                            gm = fmaxf(fmaxf(wmax[(x * 4 + q) * 4 + 0], wmax[(x * 4 + q) * 4 + 1]),
                                       fmaxf(wmax[(x * 4 + q) * 4 + 2], wmax[(x * 4 + q) * 4 + 3]));
                            gm = (jj == 0) ? INFINITY : (gm - lambda_log2) * kLn2;
                            named_bar_sync(1 + x, 128);
                        }
                        if (grp_leader && grp_valid) {
                            if (a.skip_mask) a.skip_mask[tile_row + jj] = skip_s ? 1 : 0;
                            if (want_margin) a.margin[tile_row + jj] = gm;
                        }
                    }
                    if (skip_s) {
                        if (grp_leader && grp_valid) ++n_skip;
                        continue;                            // a7: this decision tile leaves m, l, O untouched
                    }
                    if (grp_leader && grp_valid) ++n_exec;
                    if (kept == 0u) {
                        // first retained sub-tile: the MMA tile is kept -- tell the issuer and the V warp now
                        tc_fence_before();
                        if (lane == 0) {
                            votes[(x * 4 + q) * 4 + w] = (j << 2) | 2;
                            mbar_arrive(dec(x, q));
                        }
                        __syncwarp();
                        if (spec) {                          // a speculative S_x(j+1) is in flight over these columns
                            mbar_wait(s_full(x), sfpar);
                            sfpar ^= 1u;
                            tc_fence_after();
                        }
                    }
                    kept |= 1u << s;
                    m_true = fmaxf(m_true, ms);
                    if (!did_exp) exp_sub();
                    acc2 = add_f32x2(acc2, rs2);
                    dirty = true;
                    if (s == SUB / 2 - 1) {
                        // the first half of the keys is done and something in it was retained: hand it over now, so
                        // that its P V steps run while the second half is decided and exponentiated
                        if (w == 0 && lane == 0) st_shared_u32(sbase + L::kPvMaskOff + (x * 4 + q) * 4, kept);
                        tmem_wait_st();
                        tc_fence_before();
                        mbar_arrive(p_half(x));
                        half_sent = true;
                    }
                }
                prev_skip = kept == 0u;
                if (kept == 0u) {                            // every sub-tile skipped: the MMA tile is skipped
                    tc_fence_before();
                    if (lane == 0) {
                        votes[(x * 4 + q) * 4 + w] = (j << 2) | 1;
                        mbar_arrive(dec(x, q));
                    }
                    __syncwarp();
                    continue;
                }
                if (w == 0 && lane == 0) st_shared_u32(sbase + L::kPvMaskOff + (x * 4 + q) * 4, kept);
                tmem_wait_st();
                tc_fence_before();
                if (!half_sent) mbar_arrive(p_half(x));      // (release: the mask above is visible to the issuer)
                mbar_arrive(p_ready(x));
                fold();                                      // statistics for the next tile, behind the hand-over
                continue;
            }
            // ---- predicate and all-rows vote (a4)
            bool skip_grp = false, keep_any = true;
            float grp_margin = INFINITY;
            if (kSparse) {
                // votes[x][j & 3][w] = (j << 2) | (1: every row of warp w is below the threshold, 2: some row is not).
                // The MMA warp combines the four votes itself (barrier dec, one arrival per warp), so an all-skip
                // decision reaches the tensor pipe without the four warps first synchronising with each other.
                const float ref = (mode == kModeFixed) ? m_true : lse2;
                const float t2 = mhat2 - ref;                // Eq. 5 in log2 units (+inf at j = 0: tile 0 is kept)
                bool row_skip = (j > 0) && (!row_valid || (t2 < lambda_log2));
                if (mode == kModeMask) row_skip = mask_skip; // decisions read from the bitmap (one byte per decision tile)
                const bool wskip = __all_sync(0xffffffffu, row_skip);
                const int q = j & 3;
                volatile int* vt = votes + (x * 4 + q) * 4;     // ring of 4 tiles (see dec)
                tc_fence_before();                           // S_x(j) is in registers: the MMA warp may overwrite it
                if (lane == 0 && !(DSA_EXP & 8)) {
                    vt[w] = (j << 2) | (wskip ? 1 : 2);
                    mbar_arrive(dec(x, q));
                }
                __syncwarp();
                if (w == 0) { TRACE(8) }
                if (kDebug) {
                    if (want_margin) {
                        float tm = row_valid ? t2 : -INFINITY;
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) tm = fmaxf(tm, __shfl_xor_sync(0xffffffffu, tm, o));
                        if (lane == 0) wmax[(x * 4 + q) * 4 + w] = tm;
                    }
                    named_bar_sync(1 + x, 128);
                    const bool s0 = (vt[0] & 3) == 1, s1 = (vt[1] & 3) == 1, s2 = (vt[2] & 3) == 1, s3 = (vt[3] & 3) == 1;
                    if (G == 1) {
                        skip_grp = s0 && s1 && s2 && s3;
                        keep_any = !skip_grp;
                        if (want_margin)
                            grp_margin = fmaxf(fmaxf(wmax[(x * 4 + q) * 4 + 0], wmax[(x * 4 + q) * 4 + 1]),
                                               fmaxf(wmax[(x * 4 + q) * 4 + 2], wmax[(x * 4 + q) * 4 + 3]));
                    } else {
                        skip_grp = grp ? (s2 && s3) : (s0 && s1);
                        keep_any = !(s0 && s1 && s2 && s3);
                        if (want_margin)
                            grp_margin = fmaxf(wmax[(x * 4 + q) * 4 + 2 * grp], wmax[(x * 4 + q) * 4 + 2 * grp + 1]);
                    }
                    if (want_margin) grp_margin = (j == 0) ? INFINITY : (grp_margin - lambda_log2) * kLn2;
                    named_bar_sync(1 + x, 128);              // wmax / votes are reused by the next tile
                } else if (!wskip) {
                    skip_grp = false;                        // a row of this warp keeps the tile: no need to wait
                    keep_any = true;
                } else {
                    // every row of this warp is below the threshold: wait (hardware-suspended, no shared-memory
                    // polling) until all four warps have voted on tile j, then read the four votes at once
                    mbar_wait(dec(x, q), (j >> 2) & 1);
                    const int tag_keep = (j << 2) | 2;
                    const int4 v4 = lds128_volatile(sbase + L::kVotesOff + (x * 4 + q) * 16);
                    const bool k0 = v4.x == tag_keep, k1 = v4.y == tag_keep, k2 = v4.z == tag_keep, k3 = v4.w == tag_keep;
                    keep_any = k0 | k1 | k2 | k3;
                    if (G == 1) skip_grp = !keep_any;
                    else skip_grp = !((w >> 1) ? (k2 | k3) : (k0 | k1));
                }
            }
            if (grp_leader && grp_valid) {                   // a9 + optional parity outputs
                if (skip_grp) ++n_skip; else ++n_exec;
                if (kDebug) {
                    if (a.skip_mask) a.skip_mask[tile_row + j] = skip_grp ? 1 : 0;
                    if (want_margin) a.margin[tile_row + j] = grp_margin;
                }
            }
            if (w == 0) { TRACE(9) }
            PROF_TICK(4)
            prev_skip = kSparse && !keep_any;
            if (kSparse && !keep_any) {                      // a7: skipped -- m, l, O untouched
                PROF_TICK(5)
                continue;
            }
            if (spec) {
                // tile j is kept although a speculative S_x(j+1) is being written over S_x: let that MMA finish before
                // P_x goes into the same columns (the MMA warp issues S_x(j+1) again after P_x V_j)
                mbar_wait(s_full(x), sfpar);
                sfpar ^= 1u;
                tc_fence_after();
            }

            float rs0 = 0.f, rs1 = 0.f;                      // this tile's row sum, two chains
            if (kSparse && G == 2 && skip_grp) {
                // this half skipped but its partner half kept: contribute P = 0, statistics untouched
                uint32_t z[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) z[i] = 0u;
#pragma unroll
                for (int c = 0; c < BC / 32; ++c) tmem_st_x16(tS + c * 16, z);
                tmem_wait_st();
                tc_fence_before();
                mbar_arrive(p_half(x));
            } else {
                // ---- online softmax update (a5)
                if (j == 0) {
                    m_used = mhat2;
                } else {
                    const bool need = mhat2 > m_used + kRescaleThreshold;
                    if (__any_sync(0xffffffffu, need)) {
                        const float alpha = need ? fast_exp2(m_used - mhat2) : 1.f;
                        if (need) m_used = mhat2;
                        l *= alpha;
#pragma unroll
                        for (int c = 0; c < D / 32; ++c) {   // O_r *= alpha (PV of tile j-1 has completed: s_full(j))
                            uint32_t o[32];
                            tmem_ld_x32(tO + c * 32, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                            tmem_st_x32(tO + c * 32, o);
                        }
                    }
                }
                m_true = fmaxf(m_true, mhat2);
                // Warps w of the two slots share one scheduler, hence one MUFU pipe.  Two exp phases run side by side
                // both finish late; one after the other, the first finishes early and the second no later.  More
                // important, with one MMA issuer per slot a free-running pair of slots settles in phase (both in
                // softmax, then both in MMA), which idles the tensor pipe half of the time.  A warp therefore starts its
                // exp phase only when its partner is not inside one (a flag per warp, checked then set: no atomics, a
                // rare double entry is harmless).  That shifts the slots into anti-phase.  Scheduling only.
                if (kUseExpLock && nX == 2) {
                    while (ld_shared_u32(sbase + L::kLockOff + 4 * ((1 - x) * 4 + w)) != 0u) { }
                    st_shared_u32(sbase + L::kLockOff + 4 * (x * 4 + w), 1u);
                }
                TRACE(16 + w)
                const float neg_m = -m_used;
#if DSA_F32X2
                // x = s * scale - m for two logits per FFMA2, row sums as one packed pair per FADD2
                const uint64_t scale2 = pack_f32x2(scale_log2, scale_log2);
                const uint64_t negm2 = pack_f32x2(neg_m, neg_m);
                uint64_t rs2 = pack_f32x2(0.f, 0.f);
#pragma unroll
                for (int c = 0; c < BC / 32; ++c) {          // 32 columns -> 16 packed bf16x2 -> P columns [16c, 16c+16)
                    uint32_t pk[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        float x0, x1;
                        unpack_f32x2(fma_f32x2(pack_f32x2(__uint_as_float(su[c][2 * i]), __uint_as_float(su[c][2 * i + 1])),
                                               scale2, negm2), x0, x1);
                        const float p0 = fast_exp2(x0);
                        const float p1 = fast_exp2(x1);
                        rs2 = add_f32x2(rs2, pack_f32x2(p0, p1));
                        pk[i] = pack_bf16x2(p0, p1);
                    }
                    tmem_st_x16(tS + c * 16, pk);
                    if (c == BC / 64 - 1) {                  // first half of P_X is in TMEM: its P V MMAs may start
                        tmem_wait_st();
                        tc_fence_before();
                        mbar_arrive(p_half(x));
                        TRACE(20 + w)
                    }
                }
                unpack_f32x2(rs2, rs0, rs1);
#else
#pragma unroll
                for (int c = 0; c < BC / 32; ++c) {          // 32 columns -> 16 packed bf16x2 -> P columns [16c, 16c+16)
                    uint32_t pk[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const float x0 = fmaf(__uint_as_float(su[c][2 * i]), scale_log2, neg_m);
                        const float x1 = fmaf(__uint_as_float(su[c][2 * i + 1]), scale_log2, neg_m);
                        const float p0 = fast_exp2(x0);
                        const float p1 = fast_exp2(x1);
                        rs0 += p0;
                        rs1 += p1;
                        pk[i] = pack_bf16x2(p0, p1);
                    }
                    tmem_st_x16(tS + c * 16, pk);
                    if (c == BC / 64 - 1) {                  // first half of P_X is in TMEM: its P V MMAs may start
                        tmem_wait_st();
                        tc_fence_before();
                        mbar_arrive(p_half(x));
                        TRACE(20 + w)
                    }
                }
#endif
                if (kUseExpLock && nX == 2) st_shared_u32(sbase + L::kLockOff + 4 * (x * 4 + w), 0u);
            }
#undef S_AT
            PROF_TICK(6)
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(p_ready(x));
            TRACE(24 + w)
            // the statistics are updated after P has been handed over: the tail of the row-sum chain and the log2
            // must not sit between the last exp and the arrive (in-order issue would stall the arrive on them)
            if (!(kSparse && G == 2 && skip_grp)) {
                l += rs0 + rs1;
                if (kSparse && mode != kModeFixed && !(DSA_EXP & 16)) lse2 = m_used + fast_log2(l);
            }
            PROF_TICK(7)
        }
        PROF_FLUSH(8 + 8 * x, 8, r == 0)

        // ---- epilogue (a8): O / l -> bf16, lse = ln(l) + m over retained tiles
        mbar_wait(o_full(x), 0);
        tc_fence_after();
        const float inv_l = 1.f / l;
        __nv_bfloat16* orow = a.out + (static_cast<size_t>(bh) * a.N + (row_valid ? grow : 0)) * D;
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
            uint32_t o[32];
            tmem_ld_x32(tO + c * 32, o);
            tmem_wait_ld();
            if (row_valid && !kMass) {                      // (the mass kernel has no output rows)
                uint4* dst = reinterpret_cast<uint4*>(orow + c * 32);
#pragma unroll
                for (int v4 = 0; v4 < 4; ++v4) {
                    uint4 u;
                    u.x = pack_bf16x2(__uint_as_float(o[v4 * 8 + 0]) * inv_l, __uint_as_float(o[v4 * 8 + 1]) * inv_l);
                    u.y = pack_bf16x2(__uint_as_float(o[v4 * 8 + 2]) * inv_l, __uint_as_float(o[v4 * 8 + 3]) * inv_l);
                    u.z = pack_bf16x2(__uint_as_float(o[v4 * 8 + 4]) * inv_l, __uint_as_float(o[v4 * 8 + 5]) * inv_l);
                    u.w = pack_bf16x2(__uint_as_float(o[v4 * 8 + 6]) * inv_l, __uint_as_float(o[v4 * 8 + 7]) * inv_l);
                    dst[v4] = u;
                }
            }
        }
        if (a.lse && row_valid && !kMass) a.lse[static_cast<size_t>(bh) * a.N + grow] = (m_used + log2f(l)) * kLn2;
        if (a.stats && grp_leader && grp_valid) {
            atomicAdd(a.stats + 2 * bh + 0, static_cast<unsigned long long>(n_exec));
            atomicAdd(a.stats + 2 * bh + 1, static_cast<unsigned long long>(n_skip));
        }
        }
    }

    // ------------------------------------------------------------------ teardown
    tc_fence_before();
    __syncthreads();
    if (warp == kMmaWarp0) tmem_dealloc(tmem_base, kTmemCols);
}

}  // namespace dsa
