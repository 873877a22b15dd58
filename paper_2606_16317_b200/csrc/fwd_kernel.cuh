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
//   warp  9     tcgen05.mma issuer of slot 0 (one elected lane) and TMEM owner
//   warp  10    TMA producer for the V ring: slot j % NV holds V_j.  DENSE: every tile.  Sparse modes: this warp
//               reads both slots' votes on tile j and fetches V_j only if some slot keeps tile j (plus V_{j+1} ahead
//               of its votes unless the last two tiles were skipped by both slots); an unneeded tile completes its
//               ring phase without a load
//   warp  11    tcgen05.mma issuer of slot 1
// One issuer warp per slot: a thread that issues tcgen05.mma is held until its last MMA has been dispatched to the
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
constexpr int kRegsLaunch = 168;
constexpr int kRegsSoftmax = 208;
constexpr int kRegsOther = 88;
static_assert((kRegsLaunch - kRegsOther) * 128 >= (kRegsSoftmax - kRegsLaunch) * 256, "setmaxnreg pool imbalance");
constexpr int kTmemCols = 512;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
// lazy rescale: O and l are only rescaled when the row max grew by more than 2^8 (log2 domain).
constexpr float kRescaleThreshold = 8.0f;
// Of every 16 pairs of logits (one 32-column chunk), this many take their exponential on the FMA pipe (range
// reduction + cubic, packed f32x2) instead of MUFU.EX2: the MUFU pipe (16 / clk / SM) needs exactly as long for the
// N^2 exponentials as the tensor pipe for the MMAs, so every exponential moved off it shortens the softmax phase.
// Measured on config 1 (steady clocks): 0 / 2 / 3 / 4 of 16 -> DENSE 10.54 / 10.30 / 10.28 / 10.28 ms, FIXED 10.79 / 10.22 /
// 10.44 / 10.52 ms; 8 of 16 is slower than none (issue slots).
#ifndef DSA_POLY_PAIRS
#define DSA_POLY_PAIRS 2                                      // (build-time override for sweeps: -DDSA_POLY_PAIRS=n)
#endif
constexpr int kPolyPairs = DSA_POLY_PAIRS;
static_assert(kPolyPairs >= 0 && kPolyPairs <= 16, "pairs per chunk on the FMA pipe");

struct FwdArgs {
    __nv_bfloat16* out;          // [BH, N, D]
    float* lse;                  // [BH, N] or null
    unsigned long long* stats;   // [BH, 2] or null (pre-zeroed)
    uint8_t* skip_mask;          // [BH, T_r, T_c_dec] or null
    float* margin;               // [BH, T_r, T_c_dec] or null
    const float* lse_in;         // MASS mode: dense lse [BH, N], natural log
    float* mass_out;             // MASS mode: [BH, T_r, T_c] fp32, pre-zeroed: sum over the tile of e^(S - lse)
    float* sqmass_out;           // MASS mode: optional [BH, T_r, T_c] fp32, pre-zeroed: sum over the tile of e^(2 (S - lse))
    const uint8_t* mask_in;      // MASK mode: [BH, T_r, T_c] bytes, non-zero = skip (tile 0 is kept regardless)
    unsigned long long* cycles;  // debug builds: {sum of clock64 cycles per CTA, CTAs} or null (pre-zeroed)
    int N;
    int T_r;                     // decision tiles along queries
    int T_c;                     // K tiles of BC keys (MMA tiles)
    int T_c_dec;                 // decision tiles along keys: ceil(N / tile_k), = T_c unless tile_k < BC
    int n_mma_tiles;             // ceil(N / 128)
    int mode;
    float scale_log2;            // softmax_scale * log2(e)
    float lambda_log2;           // lambda * log2(e)
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
    // CTA-wide barriers (8 B each): q_full[2] k_full[NK] k_empty[NK] v_full[NV] v_empty[NV]
    static constexpr int kNumCtaBars = 2 + 2 * NK + 2 * NV;
    static constexpr int kMiscOff = kBarOff + 8 * kNumCtaBars;          // tmem_ptr (4) | pad (4) | prog[2] (8)
    // Per-slot block: everything one softmax warpgroup and its issuer exchange sits at a constant offset from ONE
    // base address per slot, which the softmax threads keep in a register for the whole K loop.
    static constexpr int kSlotOff = kMiscOff + 16;
    static constexpr int kSFull = 0;        // S_X(j) complete in TMEM                                  (count 1)
    static constexpr int kPReady = 8;       // all of P_X written (kept tiles only)                    (count 128)
    static constexpr int kOFull = 16;       // last P V of slot X complete                             (count 1)
    static constexpr int kSRead = 24;       // the 4 warps of slot X hold S_X(j) in registers          (count 4)
    static constexpr int kPPart = 32;       // p_part[3]: the first 1, 2, 3 parts of P_X written (kept tiles only; count 128)
    static constexpr int kDec = 56;         // dec[4]: the 4 warps of slot X have voted on tile j      (count 4), ring j & 3
    static constexpr int kVotes = 96;       // votes[4][4]: vote_word() of warp w on tile j, ring j & 3, 16-B rows
    static constexpr int kWmax = 160;       // wmax[4][4]: per-warp max of t (debug margins), ring j & 3
    static constexpr int kPvMask = 224;     // pvmask[4]: kept sub-tiles of tile j (SUB > 1), ring j & 3
    static constexpr int kPre = 240;        // pre[5][4] (SUB > 1): per-warp sub-tile votes: groups 0, 1 the preliminary
                                            // round of tile j (by parity), groups 2..4 the later rounds of sub-tiles 1..3
    static constexpr int kSlotStride = 320;
    static constexpr int kTotal = kSlotOff + 2 * kSlotStride;
    static constexpr int kDynamicBytes = kTotal + 1024;  // slack for the 1024-B alignment of the swizzled tiles
    static_assert(kSlotOff % 16 == 0 && kSlotStride % 16 == 0, "vote rows are read with 16-byte loads");
    static_assert(kDynamicBytes <= 232448, "exceeds the 227 KB of shared memory a CTA may use");
};

// 2^x for two logits on the FMA pipe (the MUFU-free path of the exp phase): x = n + f with n = round(x) taken from
// the low mantissa bits of x + 1.5 * 2^23, 2^f by a cubic (minimax on [-0.5, 0.5], relative error 7.5e-5: below the
// 2^-9 of the bf16 rounding of P that follows), 2^n by adding n to the exponent field.  x is clamped to >= -126.
__device__ __forceinline__ void exp2_poly_x2(uint64_t X, float& p0, float& p1) {
    float x0, x1;
    unpack_f32x2(X, x0, x1);
    const uint64_t Xc = pack_f32x2(fmaxf(x0, -126.f), fmaxf(x1, -126.f));
    const uint64_t T = add_f32x2(Xc, pack_f32x2(12582912.f, 12582912.f));
    const uint64_t Nf = add_f32x2(T, pack_f32x2(-12582912.f, -12582912.f));
    const uint64_t F = fma_f32x2(Nf, pack_f32x2(-1.f, -1.f), Xc);
    uint64_t P = fma_f32x2(pack_f32x2(0.05517167f, 0.05517167f), F, pack_f32x2(0.24261114f, 0.24261114f));
    P = fma_f32x2(P, F, pack_f32x2(0.69326097f, 0.69326097f));
    P = fma_f32x2(P, F, pack_f32x2(0.99992806f, 0.99992806f));
    float f0, f1, t0, t1;
    unpack_f32x2(P, f0, f1);
    unpack_f32x2(T, t0, t1);
    p0 = __int_as_float(__float_as_int(f0) + (__float_as_int(t0) << 23));
    p1 = __int_as_float(__float_as_int(f1) + (__float_as_int(t1) << 23));
}

// a5 for 32 columns of one row: P = 2^(s * scale - m) -> 16 packed bf16x2, row sum into the packed pair rs2.
// kPoly = the number of the chunk's 16 pairs that take the FMA-pipe polynomial (evenly spread among the MUFU ones).
template <int kPoly = kPolyPairs>
__device__ __forceinline__ void exp_chunk(const uint32_t (&s)[32], uint64_t scale2, uint64_t negm2, uint64_t& rs2,
                                          uint32_t (&pk)[16]) {
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const uint64_t X = fma_f32x2(pack_f32x2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])), scale2, negm2);
        float p0, p1;
        if (((i + 1) * kPoly) / 16 > (i * kPoly) / 16) {                        // kPoly of the 16 pairs, evenly spread
            exp2_poly_x2(X, p0, p1);
        } else {
            float x0, x1;
            unpack_f32x2(X, x0, x1);
            p0 = fast_exp2(x0);
            p1 = fast_exp2(x1);
        }
        rs2 = add_f32x2(rs2, pack_f32x2(p0, p1));
        pk[i] = pack_bf16x2(p0, p1);
    }
}

// Vote word of warp w of a slot on K tile j (ring j & 3): the tile index as a tag, the per-warp sub-tile bits of the
// narrow decision tiles (SUB > 1: bit s = "sub-tile s passes the preliminary test", bit SUB + s = "kept for certain"), and
// the warp's vote on the whole MMA tile: 1 = every row of the warp is below the threshold, 2 = some row is not.
__device__ __forceinline__ uint32_t vote_word(int j, uint32_t vote, uint32_t sub_bits = 0u) {
    return (static_cast<uint32_t>(j) << 10) | (sub_bits << 2) | vote;
}
__device__ __forceinline__ bool vote_keeps(int word, int j) {          // a keep vote on tile j (and not a stale word)
    return (static_cast<uint32_t>(word) & ~0x3fcu) == ((static_cast<uint32_t>(j) << 10) | 2u);
}
__device__ __forceinline__ bool any_vote_keeps(const int4& v, int j) {
    return vote_keeps(v.x, j) | vote_keeps(v.y, j) | vote_keeps(v.z, j) | vote_keeps(v.w, j);
}
// Speculative Q K^T of the next tile starts once this many tiles in a row were skipped.  A tile retained after a
// speculated one costs the slot a wasted Q K^T and its re-issue (~ 900 cycles); with scattered skips (the contract
// generators: 12 % sparsity, runs of length 1) speculating after ONE skipped tile ate everything the skip had saved.
constexpr int kSpecRun = 2;

// kSparse = false compiles the DENSE mode only (no predicate, no vote, V always fetched);
// kDebug adds the optional skip_mask_out / margin_out parity outputs.
// SUB == 0: the block-mass kernel of sparse_attn_block_mass (its own instantiation, so that the forward kernels carry none
// of its code: a run-time branch for it inside the sparse kernels cost them 7-9 %).
// SUB > 1 (sparse modes, G = 1): the decision tile is BR x (BC / SUB) keys -- SUB decisions per MMA tile, equal to the
// rule applied in ascending key order with the statistics updated after every retained one (block size
// 32), taken in at most two vote rounds per MMA tile (see the SUB > 1 block of the softmax warpgroups).
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
    // P_X is handed to the issuer in kHand parts of BC / kHand keys, so that the P V steps of a part run while the next
    // part is exponentiated and only the last part's steps follow the last exponential
    constexpr int kHand = (BC / 32 >= 4) ? 4 : 2;
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
    // per-slot block (see SmemLayout).  dec / votes are rings of 4 indexed by j & 3: the votes are read by the slot's
    // MMA warp, by the V warp and by the slot's own all-skip warps.  Slot x can only vote on tile j + 3 after its MMA
    // warp has finished tile j + 1, which waits for v_full of tile j + 1, which the V warp completes only after it has
    // read every vote on tile j: a ring of 4 can never be lapped.
    auto slot = [&](int x) { return sbase + L::kSlotOff + static_cast<uint32_t>(x) * L::kSlotStride; };
    const uint32_t prog0 = sbase + L::kMiscOff + 8;                  // prog[2]: tiles finished by each issuer (gate)
    volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(smem + L::kMiscOff);

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
            const uint32_t sb = slot(x);
            mbar_init(q_full(x), 1);
            mbar_init(sb + L::kSFull, 1);
            for (int h = 0; h < 3; ++h) mbar_init(sb + L::kPPart + 8 * h, 128);
            mbar_init(sb + L::kPReady, 128);
            mbar_init(sb + L::kOFull, 1);
            mbar_init(sb + L::kSRead, 4);
            for (int q = 0; q < 4; ++q) mbar_init(sb + L::kDec + 8 * q, 4);
            for (int i = 0; i < 16; ++i) st_shared_u32(sb + L::kVotes + 4 * i, 0xffffffffu);
        }
        // a K stage is released by one softmax lane per active slot (when S_x of that tile is complete),
        // a V slot by the MMA warp of every active slot (after its P V, or at once if it skipped the tile)
        for (int s = 0; s < NK; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), nX); }
        for (int s = 0; s < NV; ++s) { mbar_init(v_full(s), 1); mbar_init(v_empty(s), nX); }
        st_shared_u32(prog0, 0u);
        st_shared_u32(prog0 + 4, 0u);
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
    long long cta_t0 = 0;                                    // (debug builds: SM cycles of this CTA, for the effective clock)
    if (kDebug && threadIdx.x == 0 && a.cycles) cta_t0 = clock64();

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
                const int vs = j % NV;
                wait_slot_free(j);
                if (elect_one_sync()) {
                    mbar_arrive_expect_tx(v_full(vs), L::kKVStageBytes);
                    for (int h = 0; h < kSubD; ++h)
                        tma_load_3d(v_smem + vs * L::kKVStageBytes + h * L::kSubKVBytes, &tm_v, h * 64, j * BC, bh,
                                    v_full(vs));
                }
                __syncwarp();
            };
            if (!kSparse) {
                for (int j = 0; j < T_c; ++j) load_v(j);
            } else if (kMass) {
                // block-mass kernel: every tile is voted skipped and V is never read -- no V traffic at all, every
                // v_full phase is completed with a plain arrive (the issuers still pace the ring through v_empty)
                for (int j = 0; j < T_c; ++j) {
                    wait_slot_free(j);
                    if (lane == 0) mbar_arrive(v_full(j % NV));
                    __syncwarp();
                }
            } else {
                // Sparse modes: V_j is needed iff some slot keeps tile j.  This warp reads the votes of both slots
                // (barrier dec), fetches V_j if it is needed and not yet there, and after a kept tile fetches V_{j+1}
                // ahead of its votes (decisions are strongly correlated along j); a wasted prefetch costs L2 traffic
                // only.  A tile nobody keeps completes its v_full phase with a plain arrive.
                // The prefetch also survives the first kVPrefetchSkips skipped tiles of a run: where skipped tiles are
                // scattered among kept ones (the contract generators: 12 % sparsity, short runs) a V_j fetched only after
                // its votes would expose the L2 latency on every skip -> keep transition; inside long runs nothing is fetched.
                constexpr int kVPrefetchSkips = 2;
                load_v(0);                                   // tile 0 is always kept
                bool have = true;                            // is V_j already in (or on its way to) its slot?
                int run = 0;                                 // consecutive tiles nobody kept
                for (int j = 0; j < T_c; ++j) {
                    const int q = j & 3;
                    const bool has_next = (j + 1) < T_c;
                    bool have_next = false;
                    if (has_next && have && run < kVPrefetchSkips) { load_v(j + 1); have_next = true; }   // ahead of the votes on j
                    bool keep = false;
                    for (int x = 0; x < nX; ++x) {           // act on the first keep vote, do not wait for both slots
                        mbar_wait(slot(x) + L::kDec + 8 * q, (j >> 2) & 1);
                        const int4 vt = lds128_volatile(slot(x) + L::kVotes + 16 * q);
                        keep |= any_vote_keeps(vt, j);
                        if (keep) {
                            if (!have) { load_v(j); have = true; }
                            if (has_next && !have_next) { load_v(j + 1); have_next = true; }
                        }
                    }
                    run = keep ? 0 : run + 1;
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
            // Two issuers: warp 9 drives slot 0 and warp 11 slot 1 (every mode; measured on config 1: DENSE 10.16 ms with
            // two issuers and the gate below against 10.32 ms with one issuer driving both slots in turn; without the
            // gate 11.8 ms -- DESIGN.md section 9).
            constexpr bool kGate = true;
            const int x_lo = (warp == kMmaWarp1) ? 1 : 0;
            const int x_hi = x_lo + 1;                               // this warp drives slots [x_lo, x_hi)
            if (x_lo < nX) {
            auto issue_qk = [&](int x, uint32_t kaddr) {             // S_x = Q_x K^T, one N = BC instruction per k step
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t off = (kk >> 2) * L::kSubQBytes + (kk & 3) * 32;
                    const uint32_t koff = (kk >> 2) * L::kSubKVBytes + (kk & 3) * 32;
                    umma_ss(tmem_base + x * BC, umma_smem_desc_sw128(q_smem + x * L::kQSlotBytes + off, 16, 1024),
                            umma_smem_desc_sw128(kaddr + koff, 16, 1024), kIdescQK, kk > 0);
                }
            };
            // part h of kHand: keys [h BC / kHand, (h + 1) BC / kHand); mask (SUB > 1): bit s set = decision sub-tile s was kept
            auto issue_pv = [&](int x, uint32_t vaddr, bool acc, int part, uint32_t mask = 0xffu) {
#pragma unroll
                for (int kk = part * (BC / 16 / kHand); kk < (part + 1) * (BC / 16 / kHand); ++kk) {
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
                    umma_commit(slot(x) + L::kSFull);
                }
            }
            __syncwarp();
            if (++kstage == NK) { kstage = 0; kphase ^= 1u; }
            uint32_t ppar[2] = {0u, 0u};                 // parity of p_half / p_ready: they advance on kept tiles only
            int skip_run[2] = {0, 0};                    // tiles in a row slot x has skipped, up to tile j-1
            // Sparse modes, speculation: inside a run of skipped tiles (kSpecRun or more in a row) the next S_x(j+1) =
            // Q_x K_{j+1}^T is issued as soon as the softmax warps hold S_x(j) in registers (barrier s_read), without waiting for their vote:
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
                    const uint32_t sb = slot(x);
                    const bool spec = kSparse && skip_run[x] >= kSpecRun && has_next;
                    if (spec) {
                        mbar_wait(sb + L::kSRead, j & 1);
                        tc_fence_after();
                        if (elect_one_sync()) {
                            issue_qk(x, kaddr);
                            umma_commit(sb + L::kSFull);
                        }
                        __syncwarp();
                    }
                    bool keep = true;
                    if (kSparse) {
                        const int q = j & 3;
                        mbar_wait(sb + L::kDec + 8 * q, (j >> 2) & 1);   // all 4 warps of slot x have voted on tile j
                        tc_fence_after();                                // (their votes follow their tcgen05.ld of S_x(j))
                        const int4 vt = lds128_volatile(sb + L::kVotes + 16 * q);
                        keep = any_vote_keeps(vt, j);
                        skip_run[x] = keep ? 0 : skip_run[x] + 1;
                    }
                    if (kGate && nX == 2 && keep) {
                        // two issuers: the P V phases of two slots that both keep their tiles still take turns in the
                        // order (0, j), (1, j), (0, j+1), ... as they would with one issuer, which holds the slots in
                        // anti-phase (softmax of one under the MMAs of the other); a slot that skips never waits, and
                        // the speculative issues above run side by side.  Scheduling only.
                        const int need = (x == 0) ? j : j + 1;
                        while (static_cast<int>(ld_shared_u32(prog0 + 4 * (1 - x))) < need) { }
                    }
                    if (keep) {
#pragma unroll
                        for (int h = 0; h < kHand - 1; ++h) {
                            mbar_wait(sb + L::kPPart + 8 * h, ppar[x]);
                            if (h == 0) mbar_wait(v_full(vslot), vph);   // V_j has landed (sparse modes: fetched by the V warp
                            tc_fence_after();                            // once some slot voted to keep tile j, or prefetched)
                            uint32_t pvmask = 0xffu;
                            if (SUB > 1) pvmask = ld_shared_u32(sb + L::kPvMask + 4 * (j & 3));
                            if (elect_one_sync()) issue_pv(x, vaddr, j > 0 || h > 0, h, pvmask);
                            __syncwarp();
                        }
                        mbar_wait(sb + L::kPReady, ppar[x]);
                        tc_fence_after();
                        ppar[x] ^= 1u;
                        uint32_t pvmask2 = 0xffu;            // the mask is complete once all of P_x has been handed over
                        if (SUB > 1) pvmask2 = ld_shared_u32(sb + L::kPvMask + 4 * (j & 3));
                        if (elect_one_sync()) {
                            issue_pv(x, vaddr, true, kHand - 1, pvmask2);
                            umma_commit(v_empty(vslot));     // this slot's P_x V_j has read V_j
                            if (has_next) {
                                issue_qk(x, kaddr);          // (again, if a speculative one was overwritten by P_x)
                                umma_commit(sb + L::kSFull);
                            } else {
                                umma_commit(sb + L::kOFull);
                            }
                        }
                        __syncwarp();
                    } else {
                        if (!spec) {
                            if (elect_one_sync()) {
                                if (has_next) {
                                    issue_qk(x, kaddr);
                                    umma_commit(sb + L::kSFull);
                                } else {
                                    umma_commit(sb + L::kOFull);
                                }
                            }
                            __syncwarp();
                        }
                        // the V warp has dealt with tile j (and a prefetched but unused V_j has landed): release the slot
                        mbar_wait(v_full(vslot), vph);
                        if (lane == 0) mbar_arrive(v_empty(vslot));
                        __syncwarp();
                    }
                    if (kGate && nX == 2 && lane == 0) st_shared_u32(prog0 + 4 * x, static_cast<uint32_t>(j + 1));
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
        // This slot's barrier / vote block, this warp's vote word and the K-stage release ring: opaque to the compiler,
        // so that it keeps them in registers instead of re-deriving them from the shared-memory window base every tile
        // (which put ~60 instructions between the row max and the first exponential of a retained tile).
        uint32_t sb = slot(x);
        uint32_t vote_w = sb + L::kVotes + 4 * w;
        uint32_t kst = k_empty(0);                           // k_empty of the K stage of tile j (warp 0, lane 0 releases it)
        asm volatile("" : "+r"(sb), "+r"(vote_w), "+r"(kst));
        const bool lane0 = lane == 0;
        const bool k_releaser = w == 0 && lane == 0;

        // MASS mode: -lse_r in log2 units (rows beyond N contribute nothing)
        float neg_lse2 = -INFINITY;
        if (kMass && row_valid) neg_lse2 = -a.lse_in[static_cast<size_t>(bh) * a.N + grow] * kLog2e;
        float m_used = -INFINITY;   // stabiliser actually subtracted (log2 domain, may lag the true max)
        float m_gate = -INFINITY;   // m_used + kRescaleThreshold
        float m_true = -INFINITY;   // running max over retained tiles (log2 domain) -- FIXED mode reference
        float l = 0.f;              // sum over retained tiles of 2^(s - m_used)
        float lse2 = -INFINITY;     // m_used + log2(l): LSE over retained tiles, log2 domain (Eq. 6) -- DYNAMIC reference
        // Skip threshold of this row, log2 domain: the row votes "skip" iff mhat < thr, thr = reference + lambda
        // (Eq. 5: t = mhat - reference < lambda).  -inf before the first retained tile (tile 0 is kept: t = +inf);
        // rows beyond N carry lambda = +inf and never hold a tile (R9).  MASK mode: +inf / -inf from the bitmap.
        const float lam_row = row_valid ? lambda_log2 : INFINITY;
        float thr = -INFINITY;
        int n_skip = 0;             // decision tiles this (leader) thread saw skipped; executed = all - skipped
        uint32_t sfpar = 0;         // parity of s_full(x): one phase per S_x issued (two for a tile re-issued after a
                                    // mis-speculated skip)
        int skip_run = 0;           // tiles in a row this slot has skipped, up to tile j-1 (mirrors the issuer's count)

        for (int j = 0; j < T_c; ++j) {
            // MASK mode: this tile's byte is fetched before the wait for S_x(j), which hides the global-memory latency
            if (kSparse && !kMass && SUB == 1 && mode == kModeMask) {
                const bool mask_skip = (j > 0) && (!grp_valid || __ldg(a.mask_in + tile_row + j) != 0);
                thr = mask_skip ? INFINITY : -INFINITY;
            }
            mbar_wait(sb + L::kSFull, sfpar);
            sfpar ^= 1u;
            tc_fence_after();
            uint32_t su[BC / 32][32];                         // this thread's row of S_ij (fp32 bits)
#pragma unroll
            for (int c = 0; c < BC / 32; ++c) tmem_ld_x32(tS + c * 32, su[c]);
            // (under the TMEM loads) S_x(j) is complete, so this slot's Q K^T has read K_j for the last time (a
            // mis-speculated S_x(j) was consumed, and issued again, during tile j-1): release this slot's hold on the K stage
            mbar_arrive_if(kst, k_releaser);
            kst = (kst == k_empty(NK - 1)) ? k_empty(0) : kst + 8;
            tmem_wait_ld();
            // inside a run of skipped tiles the MMA warp issues S_x(j+1) as soon as S_x(j) has left TMEM
            const bool spec = kSparse && skip_run >= kSpecRun && (j + 1) < T_c;
            if (kSparse) {                                   // S_x(j) has left TMEM
                tc_fence_before();
                mbar_arrive_if(sb + L::kSRead, lane0);
            }
#define S_AT(c) __uint_as_float(su[(c) >> 5][(c) & 31])
            const int valid_cols = a.N - j * BC;             // ragged last K tile: columns beyond N are -inf
            if (valid_cols < BC) {
#pragma unroll
                for (int c = 0; c < BC; ++c)
                    if (c >= valid_cols) su[c >> 5][c & 31] = 0xff800000u;
            }
            if constexpr (kMass) {
                // Block mass of the dense attention probabilities: sum over the rows of the Q tile and the columns of the
                // K tile of p = e^(S_rc - lse_r) (the quantity Top-K / Top-P block selection ranks), and
                // optionally of p^2 (the per-tile term of Eq. 3's variance bound).  No P, no P V: the tile is
                // voted "skipped", so the issuer streams Q K^T only.  Packed FFMA2 / FADD2 chains as in the forward
                // kernel; one shared-memory exchange and one atomicAdd per (decision tile, K tile).
                const uint64_t scale2 = pack_f32x2(scale_log2, scale_log2);
                const uint64_t nl2 = pack_f32x2(neg_lse2, neg_lse2);
                const bool want_sq = a.sqmass_out != nullptr;
                uint64_t acc2 = pack_f32x2(0.f, 0.f), sq2 = pack_f32x2(0.f, 0.f);
#pragma unroll
                for (int c = 0; c < BC; c += 2) {
                    float x0, x1;
                    unpack_f32x2(fma_f32x2(pack_f32x2(S_AT(c), S_AT(c + 1)), scale2, nl2), x0, x1);
                    const uint64_t p2 = pack_f32x2(fast_exp2(x0), fast_exp2(x1));
                    acc2 = add_f32x2(acc2, p2);
                    if (want_sq) sq2 = fma_f32x2(p2, p2, sq2);
                }
                float a0, a1, q0, q1;
                unpack_f32x2(acc2, a0, a1);
                unpack_f32x2(sq2, q0, q1);
                float acc = row_valid ? a0 + a1 : 0.f;
                float sq = row_valid ? q0 + q1 : 0.f;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    acc += __shfl_xor_sync(0xffffffffu, acc, o);
                    if (want_sq) sq += __shfl_xor_sync(0xffffffffu, sq, o);
                }
                // the 4 (G = 1) or 2 (G = 2) warps of a decision tile combine through the wmax ring (one barrier), so
                // that one thread issues one atomic per tile
                const uint32_t wm = sb + L::kWmax + 16 * (j & 3);
                const uint32_t wq = sb + L::kPre + 16 * (j & 3);
                if (lane == 0) {
                    st_shared_u32(wm + 4 * w, __float_as_uint(acc));
                    if (want_sq) st_shared_u32(wq + 4 * w, __float_as_uint(sq));
                }
                named_bar_sync(1 + x, 128);
                if (lane == 0 && (w % (4 / G)) == 0 && grp_valid) {
                    float tot = 0.f, tsq = 0.f;
#pragma unroll
                    for (int i = 0; i < 4 / G; ++i) {
                        tot += __uint_as_float(ld_shared_u32(wm + 4 * (w + i)));
                        if (want_sq) tsq += __uint_as_float(ld_shared_u32(wq + 4 * (w + i)));
                    }
                    atomicAdd(a.mass_out + tile_row + j, tot);
                    if (want_sq) atomicAdd(a.sqmass_out + tile_row + j, tsq);
                }
                tc_fence_before();
                if (lane == 0) {
                    st_shared_u32(vote_w + 16 * (j & 3), vote_word(j, 1u));
                    mbar_arrive(sb + L::kDec + 8 * (j & 3));
                }
                __syncwarp();
                ++skip_run;
                continue;
            }
            float mhat2;                                     // tile-local row max (a3), log2 units
            bool spec_wait = spec;                           // a speculative S_x(j+1) must land before P_x(j) is written
            if constexpr (SUB <= 1) {
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
                mhat2 = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * scale_log2;
            }

            if constexpr (SUB > 1) {
                // ============ decision tiles of BC / SUB keys: SUB decisions per MMA tile, in key order
                constexpr int W = BC / SUB;                  // keys per decision tile (32 or 64)
                constexpr int CW = W / 32;                   // 32-key chunks (= hand-over parts of P_x) per decision tile
                const int q = j & 3;
                const int n_sub = min(SUB, a.T_c_dec - j * SUB);            // decision tiles of this MMA tile (ragged tail: fewer)
                const uint32_t valid = (1u << n_sub) - 1u;
                // Row maxima of the SUB decision tiles (a3); the max of the MMA tile is their max
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
                mhat2 = msub[0];
#pragma unroll
                for (int s = 1; s < SUB; ++s) mhat2 = fmaxf(mhat2, msub[s]);
                const float ref0 = (mode == kModeDynamic) ? lse2 : m_true;   // the reference before this MMA tile
                // ---- Vote round 1 (every MMA tile).  Every warp publishes (a) its vote on the WHOLE tile against the
                // statistics as they stand before it (thr = reference + lambda): within the tile the reference (LSE, or the
                // running max) can only grow, so t can only shrink, and a sub-tile skipped by this test is skipped by the
                // sequential rule too -- if every row of every warp is below thr the MMA tile is skipped, at the cost of a
                // tile with one decision; (b) per sub-tile, whether some row passes that test (candidates), and whether
                // some row keeps the sub-tile FOR CERTAIN: LSE' <= log2(2^LSE + BC 2^mhat) (DYNAMIC), m' <= max(m, mhat)
                // (FIXED) bound how far the reference of a row can grow inside the tile, whatever is retained; a row whose
                // max stays >= thr even against that bound settles its sub-tile (1e-3 covers the rounding of the
                // approximate ex2 / lg2 in the running statistics).  The votes travel in the vote word the issuer and the
                // V warp read anyway (barrier dec); the four warps read all four words.
                const bool row_skip_all = mhat2 < thr;       // (rows beyond N: thr = +inf; before the first retained tile: -inf)
                const bool wsk = __all_sync(0xffffffffu, row_skip_all);
                uint32_t wc = 0u;
                if (!wsk) {
                    const float grow_ref = ((mode == kModeDynamic) ? fast_log2(1.f + static_cast<float>(BC) * fast_exp2(mhat2 - ref0))
                                                                   : fmaxf(0.f, mhat2 - ref0)) + 1e-3f;
#pragma unroll
                    for (int s = 0; s < SUB; ++s) {
                        if (!__all_sync(0xffffffffu, msub[s] < thr)) wc |= 1u << s;
                        const bool sure = (j > 0) && (msub[s] - grow_ref >= thr);
                        if (__any_sync(0xffffffffu, sure)) wc |= 1u << (SUB + s);
                    }
                }
                tc_fence_before();                           // S_x(j) is in registers: the MMA warp may overwrite it
                st_shared_u32_if(vote_w + 16 * q, vote_word(j, wsk ? 1u : 2u, wc), lane0);
                mbar_arrive_if(sb + L::kDec + 8 * q, lane0);
                mbar_wait(sb + L::kDec + 8 * q, (j >> 2) & 1);
                const int4 v4 = lds128_volatile(sb + L::kVotes + 16 * q);
                const uint32_t any = static_cast<uint32_t>(v4.x | v4.y | v4.z | v4.w);   // (same tag in all four)
                const bool tile_kept = (any & 2u) != 0u;
                const uint32_t cand = (any >> 2) & valid;    // bit s: sub-tile s passed the test of round 1
                uint32_t kept = 0u;                          // bit s: decision sub-tile s retained
                float rsum[SUB];                             // row sums of the exponentiated sub-tiles
#pragma unroll
                for (int s = 0; s < SUB; ++s) rsum[s] = 0.f;
                // The reference of a row once the sub-tiles of set h (all before s) are retained: LSE(h) = m + log2(l +
                // sum_{i in h} rsum_i), summed in key order exactly as the statistics are updated below (Eq. 6); FIXED:
                // max(m, max_{i in h} msub_i).  `wide` rows -- the tile's row max sits more than 100 log2 units above the
                // row's reference before the tile, so that sums relative to that max would leave the fp32 range -- combine
                // log-sums instead: lsub_i = msub_i + log2(sum_c 2^(s_c - msub_i)), each relative to its own sub-tile.
                bool wide = false;
                float lsub[SUB];
#pragma unroll
                for (int s = 0; s < SUB; ++s) lsub[s] = -INFINITY;
                auto ref_after = [&](int s, uint32_t h) {
                    if (mode == kModeDynamic) {
                        if (wide) {
                            float M = ref0;
#pragma unroll
                            for (int i = 0; i < SUB - 1; ++i) if (i < s && ((h >> i) & 1u)) M = fmaxf(M, lsub[i]);
                            if (M == -INFINITY) return M;
                            float acc = fast_exp2(ref0 - M);
#pragma unroll
                            for (int i = 0; i < SUB - 1; ++i) if (i < s && ((h >> i) & 1u)) acc += fast_exp2(lsub[i] - M);
                            return M + fast_log2(acc);
                        }
                        float lh = l;
#pragma unroll
                        for (int i = 0; i < SUB - 1; ++i) if (i < s && ((h >> i) & 1u)) lh += rsum[i];
                        return m_used + fast_log2(lh);
                    }
                    float ref = m_true;
#pragma unroll
                    for (int i = 0; i < SUB - 1; ++i) if (i < s && ((h >> i) & 1u)) ref = fmaxf(ref, msub[i]);
                    return ref;
                };
                if (tile_kept) {
                    if (spec) {                              // kept after all: let the speculative S_x(j+1) land first
                        mbar_wait(sb + L::kSFull, sfpar);
                        sfpar ^= 1u;
                        tc_fence_after();
                    }
                    // the stabiliser m_used follows the max of the WHOLE MMA tile (it only has to bound the exponents; a
                    // sub-tile with a large max is never skipped), so it is fixed before any P of this tile is written
                    const bool need = mhat2 > m_gate;        // (true for every row at j = 0: m_gate = -inf)
                    if (__any_sync(0xffffffffu, need)) {
                        const float alpha = need ? fast_exp2(m_used - mhat2) : 1.f;
                        if (need) { m_used = mhat2; m_gate = mhat2 + kRescaleThreshold; }
                        l *= alpha;                          // (m_used + log2 l, hence lse2, is unchanged)
                        if (j > 0) {
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
                    // Settled after round 1: the FIRST candidate is retained (nothing was retained before it in this tile,
                    // so its test of round 1 stands), and so is every candidate some row keeps for certain.  The other
                    // candidates are OPEN: their outcome depends on which earlier sub-tiles are retained (Eq. 6).
                    const uint32_t known = ((any >> (2 + SUB)) & cand) | (cand & (0u - cand));
                    const uint32_t open = cand & ~known;
                    kept = known;
                    // P_x goes to the issuer chunk by chunk (32 keys = one part), with the mask of retained sub-tiles
                    // (a clear bit: the issuer leaves that part's P V steps out).  Parts of settled sub-tiles go at once,
                    // parts of open ones after round 2.
                    auto hand_over = [&](int c) {            // (after tmem_wait_st + fence where P was written)
                        if (w == 0 && lane == 0) st_shared_u32(sb + L::kPvMask + 4 * q, kept);
                        if (c == BC / 32 - 1) mbar_arrive(sb + L::kPReady);
                        else mbar_arrive(sb + L::kPPart + 8 * c);
                    };
                    // a5 for every candidate: all of them are exponentiated in one straight pass -- an open sub-tile that
                    // round 2 skips has cost its ex2 work and nothing else (its P columns are never read)
#pragma unroll
                    for (int s = 0; s < SUB; ++s) {
                        const bool is_cand = (cand >> s) & 1u, is_known = (known >> s) & 1u;
                        if (is_cand) {
                            uint64_t rs2 = pack_f32x2(0.f, 0.f);
#pragma unroll
                            for (int c = s * CW; c < (s + 1) * CW; ++c) {
                                uint32_t pk[16];
                                exp_chunk(su[c], scale2, negm2, rs2, pk);
                                tmem_st_x16(tS + c * 16, pk);
                                if (is_known) {
                                    tmem_wait_st();
                                    tc_fence_before();
                                    hand_over(c);
                                }
                            }
                            float r0, r1;
                            unpack_f32x2(rs2, r0, r1);
                            rsum[s] = r0 + r1;
                        } else {                             // skipped in round 1 (or beyond the last key): masked out
#pragma unroll
                            for (int c = s * CW; c < (s + 1) * CW; ++c) hand_over(c);
                        }
                    }
                    if (mode == kModeDynamic && (open != 0u || kDebug)) {
                        wide = m_used - ref0 > 100.f;        // (also every row of the first tile: ref0 = -inf)
                        if (__any_sync(0xffffffffu, wide)) {
#pragma unroll
                            for (int i = 0; i < SUB - 1; ++i) {
                                if ((cand >> i) & 1u) {
                                    const float nm = -msub[i];
                                    float acc = 0.f;
#pragma unroll
                                    for (int c = i * W; c < (i + 1) * W; ++c) acc += fast_exp2(fmaf(S_AT(c), scale_log2, nm));
                                    lsub[i] = msub[i] + fast_log2(acc);
                                }
                            }
                        }
                    }
                    if (open != 0u) {
                        // ---- Vote round 2 (only where something is open): every row evaluates the rule for each open
                        // sub-tile s under every set h of retained earlier sub-tiles that is still possible, and the warps
                        // exchange the "all my rows vote skip" bits of all of them at once; the sequential rule is then
                        // resolved from the exchanged bits along the sets that actually materialise, identically in every
                        // warp: one exchange instead of one per sub-tile.
                        uint32_t bits = 0u;                  // bit (2^s - 2 + h), h a subset of {0 .. s-1}
#pragma unroll
                        for (int s = 1; s < SUB; ++s) {
#pragma unroll
                            for (int h = 0; h < (1 << s); ++h) {
                                const uint32_t below = (1u << s) - 1u;
                                // possible: h retains every settled earlier sub-tile and nothing round 1 skipped
                                const bool possible = ((open >> s) & 1u) && ((h & ~cand) == 0u) && ((h & known & below) == (known & below));
                                if (possible) {              // (uniform over the four warps)
                                    const bool rskip = msub[s] < ref_after(s, h) + lam_row;   // (rows beyond N: lam_row = +inf)
                                    if (__all_sync(0xffffffffu, rskip)) bits |= 1u << ((1 << s) - 2 + h);
                                }
                            }
                        }
                        const uint32_t ex = sb + L::kPre + 16 * (j & 1);
                        if (lane == 0) st_shared_u32(ex + 4 * w, bits);
                        named_bar_sync(1 + x, 128);
                        const int4 b4 = lds128_volatile(ex);
                        const uint32_t allskip = static_cast<uint32_t>(b4.x & b4.y & b4.z & b4.w);   // all 128 rows (R1)
#pragma unroll
                        for (int s = 1; s < SUB; ++s) {
                            if ((open >> s) & 1u) {
                                const uint32_t h = kept & ((1u << s) - 1u);          // what was actually retained before s
                                if (!((allskip >> ((1 << s) - 2 + h)) & 1u)) kept |= 1u << s;
                            }
                        }
                        tmem_wait_st();
                        tc_fence_before();
#pragma unroll
                        for (int s = 1; s < SUB; ++s) {
                            if ((open >> s) & 1u) {
#pragma unroll
                                for (int c = s * CW; c < (s + 1) * CW; ++c) hand_over(c);
                            }
                        }
                    }
                }
                if (kDebug) {
                    // parity outputs: the decision of every sub-tile and its margin g = max_r t_r - lambda, t evaluated against
                    // the reference the sequential rule saw (the retained sub-tiles before it)
                    bool moved = false;
#pragma unroll
                    for (int s = 0; s < SUB; ++s) {
                        if (s >= n_sub) break;
                        const int jj = j * SUB + s;
                        const float ref = moved ? ref_after(s, kept & ((1u << s) - 1u)) : ref0;
                        float gm = INFINITY;
                        if (want_margin) {
                            float tm = row_valid ? msub[s] - ref : -INFINITY;
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) tm = fmaxf(tm, __shfl_xor_sync(0xffffffffu, tm, o));
                            const uint32_t wm = sb + L::kWmax + 16 * q;
                            if (lane == 0) st_shared_u32(wm + 4 * w, __float_as_uint(tm));
                            named_bar_sync(1 + x, 128);
                            const int4 m4 = lds128_volatile(wm);
                            gm = fmaxf(fmaxf(__int_as_float(m4.x), __int_as_float(m4.y)),
                                       fmaxf(__int_as_float(m4.z), __int_as_float(m4.w)));
                            gm = (jj == 0) ? INFINITY : (gm - lambda_log2) * kLn2;
                            named_bar_sync(1 + x, 128);
                        }
                        if (grp_leader && grp_valid) {
                            if (a.skip_mask) a.skip_mask[tile_row + jj] = ((kept >> s) & 1u) ? 0 : 1;
                            if (want_margin) a.margin[tile_row + jj] = gm;
                        }
                        if ((kept >> s) & 1u) moved = true;
                    }
                }
                n_skip += __popc(valid & ~kept);             // a7 / a9: skipped decision tiles leave m, l, O untouched
                if (!tile_kept) {
                    ++skip_run;
                    continue;
                }
                skip_run = 0;
                // statistics for the next tile, behind the hand-over: the retained row sums in key order
#pragma unroll
                for (int s = 0; s < SUB; ++s) {
                    if ((kept >> s) & 1u) { l += rsum[s]; m_true = fmaxf(m_true, msub[s]); }
                }
                if (mode == kModeDynamic) lse2 = m_used + fast_log2(l);
                thr = ((mode == kModeDynamic) ? lse2 : m_true) + lam_row;
                continue;
            }
            // ---- predicate and all-rows vote (a4)
            bool skip_grp = false, keep_any = true, wskip = false;
            if (kSparse && SUB == 1) {                       // (SUB > 1: voted above, every sub-tile kept for certain)
                // votes[j & 3][w] = vote_word(j, 1: every row of warp w is below the threshold, 2: some row is not).
                // The MMA warp combines the four votes itself (barrier dec, one arrival per warp), so an all-skip
                // decision reaches the tensor pipe without the four warps first synchronising with each other.
                const bool row_skip = mhat2 < thr;           // Eq. 5 against this row's threshold (false at j = 0)
                wskip = __all_sync(0xffffffffu, row_skip);
                const uint32_t q16 = static_cast<uint32_t>(j & 3) << 4;
                tc_fence_before();                           // S_x(j) is in registers: the MMA warp may overwrite it
                st_shared_u32_if(vote_w + q16, vote_word(j, wskip ? 1u : 2u), lane0);
                mbar_arrive_if(sb + L::kDec + (q16 >> 1), lane0);
                if (kDebug) {
                    float grp_margin = INFINITY;
                    const uint32_t wm = sb + L::kWmax + q16;
                    if (want_margin) {
                        const float ref = (mode == kModeFixed) ? m_true : lse2;
                        float tm = row_valid ? mhat2 - ref : -INFINITY;      // t of Eq. 5 (+inf at j = 0)
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) tm = fmaxf(tm, __shfl_xor_sync(0xffffffffu, tm, o));
                        if (lane == 0) st_shared_u32(wm + 4 * w, __float_as_uint(tm));
                    }
                    named_bar_sync(1 + x, 128);
                    const int4 v4 = lds128_volatile(sb + L::kVotes + q16);
                    const bool s0 = (v4.x & 3) == 1, s1 = (v4.y & 3) == 1, s2 = (v4.z & 3) == 1, s3 = (v4.w & 3) == 1;
                    const int4 m4 = lds128_volatile(wm);
                    const float g0 = __int_as_float(m4.x), g1 = __int_as_float(m4.y), g2 = __int_as_float(m4.z),
                                g3 = __int_as_float(m4.w);
                    if (G == 1) {
                        skip_grp = s0 && s1 && s2 && s3;
                        keep_any = !skip_grp;
                        if (want_margin) grp_margin = fmaxf(fmaxf(g0, g1), fmaxf(g2, g3));
                    } else {
                        skip_grp = grp ? (s2 && s3) : (s0 && s1);
                        keep_any = !(s0 && s1 && s2 && s3);
                        if (want_margin) grp_margin = grp ? fmaxf(g2, g3) : fmaxf(g0, g1);
                    }
                    if (want_margin) grp_margin = (j == 0) ? INFINITY : (grp_margin - lambda_log2) * kLn2;
                    named_bar_sync(1 + x, 128);              // wmax / votes are reused by the next tile
                    if (grp_leader && grp_valid) {
                        if (a.skip_mask) a.skip_mask[tile_row + j] = skip_grp ? 1 : 0;
                        if (want_margin) a.margin[tile_row + j] = grp_margin;
                    }
                    wskip = false;                           // (settled above)
                }
            } else if (kDebug && grp_leader && grp_valid) {  // DENSE: nothing is skipped, every margin is +inf
                if (a.skip_mask) a.skip_mask[tile_row + j] = 0;
                if (want_margin) a.margin[tile_row + j] = INFINITY;
            }
            // ---- online softmax update (a5), first part.  A retained tile of a warp with a keeping row, outside a skip run
            // and with no row whose max grew past the lazy-rescale gate -- the common case -- takes none of the branches
            // below: one test covers the three rare events.  The first retained tile takes the rescale path too (m_used =
            // m_gate = -inf: alpha = 0, l = 0 stays 0; O, still unwritten, is overwritten by the non-accumulating P V of
            // tile 0), which spares a j == 0 test.
            const bool need = mhat2 > m_gate;
            const bool need_any = __any_sync(0xffffffffu, need);
            if (__builtin_expect(wskip || spec_wait || need_any || (kSparse && kDebug), 0)) {
                if (wskip) {
                    // every row of this warp is below the threshold: wait (hardware-suspended, no shared-memory
                    // polling) until all four warps have voted on tile j, then read the four votes at once
                    const uint32_t q16 = static_cast<uint32_t>(j & 3) << 4;
                    mbar_wait(sb + L::kDec + (q16 >> 1), (j >> 2) & 1);
                    const int4 v4 = lds128_volatile(sb + L::kVotes + q16);
                    const bool k0 = vote_keeps(v4.x, j), k1 = vote_keeps(v4.y, j), k2 = vote_keeps(v4.z, j), k3 = vote_keeps(v4.w, j);
                    keep_any = k0 | k1 | k2 | k3;
                    if (G == 1) skip_grp = !keep_any;
                    else skip_grp = !((w >> 1) ? (k2 | k3) : (k0 | k1));
                }
                if (skip_grp) ++n_skip;                      // a9
                if (kSparse && !keep_any) {                  // a7: skipped -- m, l, O untouched
                    ++skip_run;
                    continue;
                }
                if (spec_wait) {
                    // tile j is kept although a speculative S_x(j+1) is being written over S_x: let that MMA finish before
                    // P_x goes into the same columns (the MMA warp issues S_x(j+1) again after P_x V_j)
                    mbar_wait(sb + L::kSFull, sfpar);
                    sfpar ^= 1u;
                    tc_fence_after();
                }
                if (need_any && !(kSparse && G == 2 && skip_grp)) {
                    const float alpha = need ? fast_exp2(m_used - mhat2) : 1.f;
                    if (need) { m_used = mhat2; m_gate = mhat2 + kRescaleThreshold; }
                    l *= alpha;
                    if (j > 0) {
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
            }
            skip_run = 0;

            uint64_t rs2 = pack_f32x2(0.f, 0.f);             // this tile's row sum, one packed pair of chains
            if (kSparse && G == 2 && skip_grp) {
                // this half skipped but its partner half kept: contribute P = 0, statistics untouched
                uint32_t z[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) z[i] = 0u;
#pragma unroll
                for (int c = 0; c < BC / 32; ++c) tmem_st_x16(tS + c * 16, z);
                tmem_wait_st();
                tc_fence_before();
#pragma unroll
                for (int h = 0; h < kHand - 1; ++h) mbar_arrive(sb + L::kPPart + 8 * h);
            } else {
                // ---- online softmax update (a5), second part
                // x = s * scale - m for two logits per FFMA2, row sums as one packed pair per FADD2
                const float neg_m = -m_used;
                const uint64_t scale2 = pack_f32x2(scale_log2, scale_log2);
                const uint64_t negm2 = pack_f32x2(neg_m, neg_m);
#pragma unroll
                for (int c = 0; c < BC / 32; ++c) {          // 32 columns -> 16 packed bf16x2 -> P columns [16c, 16c+16)
                    uint32_t pk[16];
                    exp_chunk(su[c], scale2, negm2, rs2, pk);
                    tmem_st_x16(tS + c * 16, pk);
                    if ((c + 1) % (BC / 32 / kHand) == 0 && c + 1 < BC / 32) {   // a part of P_X is in TMEM: its P V MMAs may start
                        tmem_wait_st();
                        tc_fence_before();
                        mbar_arrive(sb + L::kPPart + 8 * ((c + 1) / (BC / 32 / kHand) - 1));
                    }
                }
            }
#undef S_AT
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(sb + L::kPReady);
            // The statistics are updated after P has been handed over: the tail of the row-sum chain, the log2 and the
            // next tile's threshold must not sit between the last exp and the arrive (in-order issue would stall the
            // arrive on them); here they run while the tensor pipe works on P_x V_j and S_x(j+1).
            if (!(kSparse && G == 2 && skip_grp)) {
                float rs0, rs1;
                unpack_f32x2(rs2, rs0, rs1);
                l += rs0 + rs1;
                if (kSparse) {
                    m_true = fmaxf(m_true, mhat2);
                    if (mode != kModeFixed) lse2 = m_used + fast_log2(l);
                    if (mode != kModeMask) thr = ((mode == kModeFixed) ? m_true : lse2) + lam_row;
                }
            }
        }

        // ---- epilogue (a8): O / l -> bf16, lse = ln(l) + m over retained tiles
        mbar_wait(sb + L::kOFull, 0);
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
        if (a.stats && grp_leader && grp_valid && !kMass) {
            // a9: every decision tile of this Q tile is either executed or skipped (DENSE: none skipped)
            atomicAdd(a.stats + 2 * bh + 0, static_cast<unsigned long long>(a.T_c_dec - n_skip));
            atomicAdd(a.stats + 2 * bh + 1, static_cast<unsigned long long>(n_skip));
        }
        }
    }

    // ------------------------------------------------------------------ teardown
    tc_fence_before();
    __syncthreads();
    if (warp == kMmaWarp0) tmem_dealloc(tmem_base, kTmemCols);
    if (kDebug && threadIdx.x == 0 && a.cycles) {
        atomicAdd(a.cycles, static_cast<unsigned long long>(clock64() - cta_t0));
        atomicAdd(a.cycles + 1, 1ull);
    }
}

}  // namespace dsa
