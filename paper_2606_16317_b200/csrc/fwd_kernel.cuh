// Tile-skipping FlashAttention forward for sm_100a (B200).
//
// Implements SURVEY.md section 8(a) steps a1-a9 / PAPER.md section 3.1 in ONE kernel, three modes:
// DENSE, FIXED (BLASST indicator) and DYNAMIC (DynSparse, Eq. 5-6).
//
// CTA = 2 MMA tiles (slots X = 0, 1) of 128 query rows of one (b, h), sharing every K_j / V_j tile:
//   warps 0-3   softmax warpgroup of slot 0 (thread <-> query row <-> TMEM lane)
//   warps 4-7   softmax warpgroup of slot 1
//   warp  8     TMA producer for Q (once) and the K ring (runs ahead of the decisions)
//   warp  9     tcgen05.mma issuer (one elected lane) and TMEM owner
//   warp  10    TMA producer for the V ring in DENSE mode (in the sparse modes the MMA warp fetches V_j itself,
//               and only if some slot keeps tile j or tile j-1 needed its V)
//   warp  11    idle (completes the third warpgroup so that setmaxnreg can hand its registers over)
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
#define TRACE(slot) if (a.prof && blockIdx.x == DSA_TRACE_CTA && blockIdx.y == 0 && j >= DSA_TRACE_J0 && j < DSA_TRACE_J0 + 32 && (threadIdx.x & 31) == 0) a.prof[(1 << 20) + ((j - DSA_TRACE_J0) * 2 + x) * 16 + (slot)] = clock64();
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

enum : int { kModeDense = 0, kModeFixed = 1, kModeDynamic = 2 };

constexpr int kNumThreads = 384;      // 3 warpgroups
constexpr int kKProducerWarp = 8;
constexpr int kMmaWarp = 9;
constexpr int kVProducerWarp = 10;
// setmaxnreg: the kernel launches with 168 registers/thread (65536 / 384); the two softmax warpgroups grow to
// 208 (a full S row lives in registers), the producer/MMA warpgroup shrinks to 88.  The registers the 128
// threads give up must cover what the 256 softmax threads take, or setmaxnreg.inc never returns.
constexpr int kRegsLaunch = 168;
constexpr int kRegsSoftmax = 208;
constexpr int kRegsOther = 88;
static_assert((kRegsLaunch - kRegsOther) * 128 >= (kRegsSoftmax - kRegsLaunch) * 256, "setmaxnreg pool imbalance");
constexpr int kTmemCols = 512;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
// lazy rescale: O and l are only rescaled when the row max grew by more than 2^8 (log2 domain).
constexpr float kRescaleThreshold = 8.0f;
// of every 16 (p0, p1) pairs of a 32-column chunk, this many are exponentiated on the FMA pipe (exp2_fma).
// Measured on B200: the softmax warps are issue-bound, not MUFU-bound, so 0 is fastest.
#ifndef DSA_EMUL_PAIRS
#define DSA_EMUL_PAIRS 0
#endif
constexpr int kEmulPairs = DSA_EMUL_PAIRS;

struct FwdArgs {
    __nv_bfloat16* out;          // [BH, N, D]
    float* lse;                  // [BH, N] or null
    unsigned long long* stats;   // [BH, 2] or null (pre-zeroed)
    uint8_t* skip_mask;          // [BH, T_r, T_c] or null
    float* margin;               // [BH, T_r, T_c] or null
    int N;
    int T_r;                     // decision tiles along queries
    int T_c;                     // decision tiles along keys (= K tiles)
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
    //                      s_full[2] p_half[2] p_ready[2] o_full[2] s_read[2] dec[2][2] vcmd[NV]
    static constexpr int kNumBars = 2 + 2 * NK + 2 * NV + 8 + 2 + 4 + NV;
    static constexpr int kMiscOff = kBarOff + 8 * kNumBars;
    // misc: tmem_ptr (4) | pad (12) | vcmd[NV] (<= 32) | votes[2][2][4] (64) | wmax[2][2][4] (64)
    static constexpr int kMiscBytes = 16 + 16 + 16 + 64 + 64;
    static constexpr int kTotal = kMiscOff + kMiscBytes;
    static constexpr int kDynamicBytes = kTotal + 1024;  // slack for the 1024-B alignment of the swizzled tiles
    static_assert(kDynamicBytes <= 232448, "exceeds the 227 KB of shared memory a CTA may use");
};

// kSparse = false compiles the DENSE mode only (no predicate, no vote, V always fetched);
// kDebug adds the optional skip_mask_out / margin_out parity outputs.
template <int D, int BC, int G, int NK, int NV, bool kSparse, bool kDebug>
__global__ void __launch_bounds__(kNumThreads, 1)
sparse_attn_fwd_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                       const __grid_constant__ CUtensorMap tm_v, const FwdArgs a) {
    using L = SmemLayout<D, BC, NK, NV>;
    static_assert(D == 64 || D == 128, "head dim");
    static_assert(BC == 64 || BC == 128, "key tile");
    static_assert(2 * BC + 2 * D <= kTmemCols, "TMEM budget");
    constexpr int BR = 128 / G;
    constexpr int kSubD = D / 64;
    constexpr uint32_t kIdescQK = umma_idesc_bf16(128, BC, 0);   // S = Q K^T: A, B both K-major
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
    // the 4 warps of slot X have voted on tile j.  One barrier per tile parity: inside a run of skipped tiles the
    // softmax warps may vote on tile j+1 (its S was issued speculatively) before the MMA warp has looked at the
    // votes of tile j, and a single barrier two phases ahead of its waiter would alias.
    auto dec = [&](int x, int par) { return bar0 + 8u * (kB + 10 + 2 * x + par); };
    auto vcmd_bar = [&](int s) { return bar0 + 8u * (kB + 14 + s); }; // sparse modes: "load V_j into slot s" posted
    volatile int* vcmd = reinterpret_cast<volatile int*>(smem + L::kMiscOff + 16);               // [NV]
    volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(smem + L::kMiscOff);
    volatile int* votes = reinterpret_cast<volatile int*>(smem + L::kMiscOff + 48);              // [2][2][4]
    volatile float* wmax = reinterpret_cast<volatile float*>(smem + L::kMiscOff + 112);          // [2][2][4]

    const int warp = threadIdx.x >> 5;
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
            mbar_init(dec(x, 0), 4);
            mbar_init(dec(x, 1), 4);
            mbar_init(s_read(x), 4);
        }
        for (int s = 0; s < NV; ++s) mbar_init(vcmd_bar(s), 1);
        for (int s = 0; s < NK; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), 1); }
        for (int s = 0; s < NV; ++s) { mbar_init(v_full(s), 1); mbar_init(v_empty(s), 1); }
        for (int i = 0; i < 16; ++i) votes[i] = -1;
        fence_mbar_init();
    }
    if (warp == kMmaWarp) {
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
            int slot = 0, nloaded = 0;
            uint32_t phase = 0;
            auto load_v = [&](int j) {
                if (nloaded >= NV) mbar_wait(v_empty(slot), phase ^ 1u);
                if (elect_one_sync()) {
                    mbar_arrive_expect_tx(v_full(slot), L::kKVStageBytes);
                    for (int h = 0; h < kSubD; ++h)
                        tma_load_3d(v_smem + slot * L::kKVStageBytes + h * L::kSubKVBytes, &tm_v, h * 64, j * BC, bh,
                                    v_full(slot));
                }
                __syncwarp();
                ++nloaded;
                if (++slot == NV) { slot = 0; phase ^= 1u; }
            };
            // Dense mode: every V_j is fetched.  Sparse modes: the MMA warp, which is the first to know a tile's
            // decision, posts "load V_j" commands (one mbarrier + one word per ring slot) and this warp executes
            // them, so that waiting for a free slot never stalls the tensor-pipe issuer.  j < 0 ends the loop.
            if (!kSparse) {
                for (int j = 0; j < T_c; ++j) load_v(j);
            } else {
                int cslot = 0;
                uint32_t cphase = 0;
                while (true) {
                    mbar_wait(vcmd_bar(cslot), cphase);
                    const int j = vcmd[cslot];
                    if (j < 0) break;
                    load_v(j);
                    if (++cslot == NV) { cslot = 0; cphase ^= 1u; }
                }
            }
        } else if (warp == kMmaWarp) {
            // ========================================================== MMA issuer (a2, a6)
            auto issue_qk = [&](int x, uint32_t kaddr, int j = 1000) {
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
#if defined(DSA_EXP) && (DSA_EXP & 8)
                    if (kk >= 4) break;
#endif
#if defined(DSA_EXP) && (DSA_EXP & 16)
                    if (kk >= 1) break;
#endif
                    const uint32_t off = (kk >> 2) * L::kSubQBytes + (kk & 3) * 32;
                    const uint32_t koff = (kk >> 2) * L::kSubKVBytes + (kk & 3) * 32;
                    umma_ss(tmem_base + x * BC, umma_smem_desc_sw128(q_smem + x * L::kQSlotBytes + off, 16, 1024),
                            umma_smem_desc_sw128(kaddr + koff, 16, 1024), kIdescQK, kk > 0);
#ifdef DSA_PROF
                    if (a.prof && blockIdx.x == DSA_TRACE_CTA && blockIdx.y == 0 && j >= DSA_TRACE_J0 && j < DSA_TRACE_J0 + 32 && (kk == 0 || kk == 7))
                        a.prof[(1 << 20) + ((j - DSA_TRACE_J0) * 2 + x) * 16 + 10 + (kk + 1) / 2] = clock64();
#endif
                }
            };
            auto issue_pv = [&](int x, uint32_t vaddr, bool acc, int half) {   // half 0 / 1: keys [0, BC/2) / [BC/2, BC)
#pragma unroll
                for (int kk = half * (BC / 32); kk < (half + 1) * (BC / 32); ++kk) {
                    // 16 keys = 16 rows of 128 B; d sub-tiles (64 columns) are L::kSubKVBytes apart (LBO)
                    umma_ts(tmem_base + 2 * BC + x * D, tmem_base + x * BC + kk * 8,
                            umma_smem_desc_sw128(vaddr + kk * 2048, L::kSubKVBytes, 1024), kIdescPV, acc || kk > 0);
                }
            };
            int kstage = 0, vslot = 0;
            uint32_t kphase = 0, vphase = 0;

            PROF_DECL(8)
            for (int x = 0; x < nX; ++x) mbar_wait(q_full(x), 0);
            mbar_wait(k_full(0), 0);
            PROF_TICK(0)
            tc_fence_after();
            if (elect_one_sync()) {
                for (int x = 0; x < nX; ++x) {
                    issue_qk(x, k_smem);
                    umma_commit(s_full(x));
                }
                umma_commit(k_empty(0));
            }
            __syncwarp();
            if (++kstage == NK) { kstage = 0; kphase ^= 1u; }

            uint32_t ppar[2] = {0u, 0u};                     // parity of p_half / p_ready: they advance on kept tiles only
            // Sparse modes.  (1) V: tile j's V is requested (from the V warp) once some slot has voted to keep tile j,
            // and V_{j+1} right after it (decisions are strongly correlated along j).  (2) Speculation: inside a run
            // of skipped tiles the next S_x(j+1) = Q_x K_{j+1}^T is issued as soon as the softmax warps hold S_x(j) in
            // registers (barrier s_read), without waiting for their vote: the vote is then off the critical chain.
            // If tile j turns out to be kept, the softmax warps let the speculative MMA finish before they write P_x
            // over it, and S_x(j+1) is issued again after P_x V_j.  Scheduling only: no decision depends on it.
            int lslot = 0;                                   // V ring, command side
            auto post_v = [&](int j) {
                if (elect_one_sync()) {
                    vcmd[lslot] = j;
                    mbar_arrive(vcmd_bar(lslot));
                }
                __syncwarp();
                if (++lslot == NV) lslot = 0;
            };
            bool v_loaded = !kSparse;                        // is V_j in (or on its way to) slot vslot?
            bool v_next = false;                             // has V_{j+1} been requested?
            bool prev_skip[2] = {false, false};              // did slot x skip tile j-1?
            if (kSparse) { post_v(0); v_loaded = true; }     // tile 0 is always kept
            for (int j = 0; j < T_c; ++j) {
                const int par = j & 1;
                const bool has_next = (j + 1) < T_c;
                bool v_waited = false;
                const uint32_t vaddr = v_smem + vslot * L::kKVStageBytes;
                const uint32_t kaddr = k_smem + kstage * L::kKVStageBytes;
                PROF_TICK(1)
                if (has_next) { mbar_wait(k_full(kstage), kphase); tc_fence_after(); }   // K_{j+1} has landed
                { const int x = 0; TRACE(11) }
                PROF_TICK(5)
                bool spec[2] = {false, false};
                if (kSparse) {
                    for (int x = 0; x < nX; ++x) {
                        spec[x] = prev_skip[x] && has_next;
                        if (spec[x]) {
                            mbar_wait(s_read(x), par);       // S_x(j) is in the softmax warps' registers
                            TRACE(12)
                            tc_fence_after();
                            if (elect_one_sync()) {
                                issue_qk(x, kaddr, j);
                                umma_commit(s_full(x));
                            }
                            __syncwarp();
                            TRACE(13)
                        }
                    }
                    PROF_TICK(6)
                }
                for (int x = 0; x < nX; ++x) {
                    bool keep = true;
#if defined(DSA_EXP) && (DSA_EXP & 2)
                    if (kSparse && spec[x]) { keep = false; } else
#endif
                    if (kSparse) {
                        TRACE(0)
                        mbar_wait(dec(x, par), (j >> 1) & 1);              // all 4 warps of slot x have voted on tile j
                        tc_fence_after();
                        TRACE(1)
                        PROF_TICK(2 + x)
                        const int tag_keep = (j << 2) | 2;
                        const int4 vt = lds128_volatile(sbase + L::kMiscOff + 48 + (x * 2 + par) * 16);
                        keep = (vt.x == tag_keep) | (vt.y == tag_keep) | (vt.z == tag_keep) | (vt.w == tag_keep);
                        prev_skip[x] = !keep;
                        if (keep) {
                            if (!v_loaded) { post_v(j); v_loaded = true; }                 // not prefetched: fetch V_j now
                            if (!v_next && has_next) { post_v(j + 1); v_next = true; }     // and prefetch V_{j+1}
                        }
                        PROF_TICK(7)
                    }
                    if (keep) {
                        mbar_wait(p_half(x), ppar[x]);
                        tc_fence_after();
                        PROF_TICK(2 + x)
                        if (!v_waited) { mbar_wait(v_full(vslot), vphase); tc_fence_after(); v_waited = true; }
                        PROF_TICK(4)
                        if (elect_one_sync()) issue_pv(x, vaddr, j > 0, 0);
                        __syncwarp();
                        PROF_TICK(1)
                        mbar_wait(p_ready(x), ppar[x]);
                        tc_fence_after();
                        ppar[x] ^= 1u;
                        PROF_TICK(2 + x)
                    }
                    TRACE(2)
                    if (keep || !spec[x]) {
                        if (elect_one_sync()) {
                            if (keep) issue_pv(x, vaddr, true, 1);
                            if (has_next) {
                                issue_qk(x, kaddr, j);       // (again, if the speculative one was overwritten by P_x)
                                umma_commit(s_full(x));
                            } else {
                                umma_commit(o_full(x));
                            }
                        }
                        __syncwarp();
                    }
                    TRACE(3)
                    PROF_TICK(1)
                }
                if (v_loaded) {                              // a V slot was filled for this tile: release it
                    if (!v_waited) mbar_wait(v_full(vslot), vphase);
                    if (elect_one_sync()) umma_commit(v_empty(vslot));
                    __syncwarp();
                    if (++vslot == NV) { vslot = 0; vphase ^= 1u; }
                }
                PROF_TICK(4)
                if (has_next) {
                    if (elect_one_sync()) umma_commit(k_empty(kstage));
                    __syncwarp();
                    if (++kstage == NK) { kstage = 0; kphase ^= 1u; }
                }
                if (kSparse) { v_loaded = v_next; v_next = false; }
            }
            if (kSparse) post_v(-1);                         // every requested V has been consumed: stop the V warp
            PROF_FLUSH(0, 8, lane == 0)
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
        const size_t tile_row = (static_cast<size_t>(bh) * a.T_r + dtile) * static_cast<size_t>(T_c);
        const int mode = a.mode;
        const float scale_log2 = a.scale_log2;
        const float lambda_log2 = a.lambda_log2;
        const bool want_margin = kDebug && a.margin != nullptr;

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
            const int par = j & 1;
            PROF_TICK(0)
            if (w == 0) { TRACE(4) }
            mbar_wait(s_full(x), sfpar);
            sfpar ^= 1u;
            tc_fence_after();
            if (w == 0) { TRACE(5) }
            PROF_TICK(1)
            uint32_t su[BC / 32][32];                         // this thread's row of S_ij (fp32 bits)
#pragma unroll
            for (int c = 0; c < BC / 32; ++c) tmem_ld_x32(tS + c * 32, su[c]);
            tmem_wait_ld();
            // inside a run of skipped tiles the MMA warp issues S_x(j+1) as soon as S_x(j) has left TMEM
            const bool spec = kSparse && prev_skip && (j + 1) < T_c;
            if (kSparse) {
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
#if defined(DSA_EXP) && (DSA_EXP & 1)
            const float mhat2 = S_AT(0) * scale_log2;
#else
            const float mhat2 = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * scale_log2;   // tile-local row max (a3)
#endif
            if (w == 0) { TRACE(7) }
            PROF_TICK(3)

            // ---- predicate and all-rows vote (a4)
            bool skip_grp = false, keep_any = true;
            float grp_margin = INFINITY;
            if (kSparse) {
                // votes[x][j & 1][w] = (j << 2) | (1: every row of warp w is below the threshold, 2: some row is not).
                // The MMA warp combines the four votes itself (barrier dec, one arrival per warp), so an all-skip
                // decision reaches the tensor pipe without the four warps first synchronising with each other.
                const float ref = (mode == kModeDynamic) ? lse2 : m_true;
                const float t2 = mhat2 - ref;                // Eq. 5 in log2 units (+inf at j = 0: tile 0 is kept)
                const bool row_skip = (j > 0) && (!row_valid || (t2 < lambda_log2));
                const bool wskip = __all_sync(0xffffffffu, row_skip);
                volatile int* vt = votes + (x * 2 + par) * 4;   // double-buffered by tile parity
                tc_fence_before();                           // S_x(j) is in registers: the MMA warp may overwrite it
                if (lane == 0) {
                    vt[w] = (j << 2) | (wskip ? 1 : 2);
                    mbar_arrive(dec(x, par));
                }
                __syncwarp();
                if (w == 0) { TRACE(8) }
                if (kDebug) {
                    if (want_margin) {
                        float tm = row_valid ? t2 : -INFINITY;
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) tm = fmaxf(tm, __shfl_xor_sync(0xffffffffu, tm, o));
                        if (lane == 0) wmax[(x * 2 + par) * 4 + w] = tm;
                    }
                    named_bar_sync(1 + x, 128);
                    const bool s0 = (vt[0] & 3) == 1, s1 = (vt[1] & 3) == 1, s2 = (vt[2] & 3) == 1, s3 = (vt[3] & 3) == 1;
                    if (G == 1) {
                        skip_grp = s0 && s1 && s2 && s3;
                        keep_any = !skip_grp;
                        if (want_margin)
                            grp_margin = fmaxf(fmaxf(wmax[(x * 2 + par) * 4 + 0], wmax[(x * 2 + par) * 4 + 1]),
                                               fmaxf(wmax[(x * 2 + par) * 4 + 2], wmax[(x * 2 + par) * 4 + 3]));
                    } else {
                        skip_grp = grp ? (s2 && s3) : (s0 && s1);
                        keep_any = !(s0 && s1 && s2 && s3);
                        if (want_margin)
                            grp_margin = fmaxf(wmax[(x * 2 + par) * 4 + 2 * grp], wmax[(x * 2 + par) * 4 + 2 * grp + 1]);
                    }
                    if (want_margin) grp_margin = (j == 0) ? INFINITY : (grp_margin - lambda_log2) * kLn2;
                    named_bar_sync(1 + x, 128);              // wmax / votes are reused by the next tile
                } else if (!wskip) {
                    skip_grp = false;                        // a row of this warp keeps the tile: no need to wait
                    keep_any = true;
                } else {
                    // every row of this warp is below the threshold: wait (hardware-suspended, no shared-memory
                    // polling) until all four warps have voted on tile j, then read the four votes at once
#if defined(DSA_EXP) && (DSA_EXP & 4)
                    if (j < 2)
#endif
                    mbar_wait(dec(x, par), (j >> 1) & 1);
                    const int tag_keep = (j << 2) | 2;
                    const int4 v4 = lds128_volatile(sbase + L::kMiscOff + 48 + (x * 2 + par) * 16);
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
                const float neg_m = -m_used;
                float rs0 = 0.f, rs1 = 0.f;
#pragma unroll
                for (int c = 0; c < BC / 32; ++c) {          // 32 columns -> 16 packed bf16x2 -> P columns [16c, 16c+16)
                    uint32_t pk[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const float x0 = fmaf(__uint_as_float(su[c][2 * i]), scale_log2, neg_m);
                        const float x1 = fmaf(__uint_as_float(su[c][2 * i + 1]), scale_log2, neg_m);
                        const bool emul = kEmulPairs >= 8 ? ((i & 1) == 1 && (i >> 1) < kEmulPairs)
                                                          : ((i & 3) == 3 && (i >> 2) < kEmulPairs);
                        const float p0 = emul ? exp2_fma(x0) : fast_exp2(x0);
                        const float p1 = emul ? exp2_fma(x1) : fast_exp2(x1);
                        rs0 += p0;
                        rs1 += p1;
                        pk[i] = pack_bf16x2(p0, p1);
                    }
                    tmem_st_x16(tS + c * 16, pk);
                    if (c == BC / 64 - 1) {                  // first half of P_X is in TMEM: its P V MMAs may start
                        tmem_wait_st();
                        tc_fence_before();
                        mbar_arrive(p_half(x));
                    }
                }
                l += rs0 + rs1;
                if (kSparse) lse2 = m_used + fast_log2(l);
            }
#undef S_AT
            PROF_TICK(6)
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(p_ready(x));
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
            if (row_valid) {
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
        if (a.lse && row_valid) a.lse[static_cast<size_t>(bh) * a.N + grow] = (m_used + log2f(l)) * kLn2;
        if (a.stats && grp_leader && grp_valid) {
            atomicAdd(a.stats + 2 * bh + 0, static_cast<unsigned long long>(n_exec));
            atomicAdd(a.stats + 2 * bh + 1, static_cast<unsigned long long>(n_skip));
        }
        }
    }

    // ------------------------------------------------------------------ teardown
    tc_fence_before();
    __syncthreads();
    if (warp == kMmaWarp) tmem_dealloc(tmem_base, kTmemCols);
}

}  // namespace dsa
