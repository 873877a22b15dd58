// Tile-skipping FlashAttention forward for sm_100a (B200).
//
// Implements SURVEY.md section 8(a) steps a1-a9 / PAPER.md section 3.1 in ONE kernel, three modes:
// DENSE, FIXED (BLASST indicator) and DYNAMIC (DynSparse, Eq. 5-6).
//
// CTA = 2 MMA tiles (slots X = 0, 1) of 128 query rows of one (b, h), sharing every K_j / V_j tile:
//   warps 0-3   softmax warpgroup of slot 0 (thread <-> query row <-> TMEM lane)
//   warps 4-7   softmax warpgroup of slot 1
//   warp  8     TMA producer: Q once, then K_0, V_0, K_1, V_1, ... through an NSTAGE mbarrier ring
//   warp  9     tcgen05.mma issuer (one elected thread) and TMEM owner
//   warps 10-11 idle (they complete the third warpgroup so that setmaxnreg can hand its registers over)
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

enum : int { kModeDense = 0, kModeFixed = 1, kModeDynamic = 2 };

constexpr int kNumThreads = 384;      // 3 warpgroups: softmax 0, softmax 1, {producer, MMA, 2 idle warps}
constexpr int kProducerWarp = 8;
constexpr int kMmaWarp = 9;
// setmaxnreg: the kernel launches with 168 registers/thread (65536 / 384); the two softmax warpgroups
// grow to 232 (a full S row lives in registers), the producer/MMA warpgroup shrinks to 40.
constexpr int kRegsSoftmax = 232;
constexpr int kRegsOther = 40;
constexpr int kTmemCols = 512;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
// lazy rescale: O and l are only rescaled when the row max grew by more than 2^8 (log2 domain).
constexpr float kRescaleThreshold = 8.0f;

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
};

template <int D, int BC, int NSTAGE>
struct SmemLayout {
    static constexpr int kQSlotBytes = 128 * D * 2;
    static constexpr int kSubQBytes = 128 * 128;        // one 64-column (128 B) sub-tile of Q
    static constexpr int kKVStageBytes = BC * D * 2;
    static constexpr int kSubKVBytes = BC * 128;        // one 64-column sub-tile of K or V
    static constexpr int kQOff = 0;
    static constexpr int kKVOff = 2 * kQSlotBytes;
    static constexpr int kBarOff = kKVOff + NSTAGE * kKVStageBytes;
    // barriers (8 B each): q_full[2], kv_full[NSTAGE], kv_empty[NSTAGE], s_full[2], p_ready[2], o_full[2]
    static constexpr int kNumBars = 2 + 2 * NSTAGE + 6;
    static constexpr int kMiscOff = kBarOff + 8 * kNumBars;
    // misc: tmem_ptr (4) | keepflag[2][2] (16) | votes[2][2][4] (64) | wmax[2][2][4] (64)
    static constexpr int kMiscBytes = 4 + 16 + 64 + 64 + 12;
    static constexpr int kTotal = kMiscOff + kMiscBytes;
    static constexpr int kDynamicBytes = kTotal + 1024;  // slack for the 1024-B alignment of the swizzled tiles
};

// kSparse = false compiles the DENSE mode only (no predicate, no vote); kDebug adds the optional
// skip_mask_out / margin_out parity outputs.
template <int D, int BC, int G, int NSTAGE, bool kSparse, bool kDebug>
__global__ void __launch_bounds__(kNumThreads, 1)
sparse_attn_fwd_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                       const __grid_constant__ CUtensorMap tm_v, const FwdArgs a) {
    using L = SmemLayout<D, BC, NSTAGE>;
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
    const uint32_t kv_smem = sbase + L::kKVOff;
    const uint32_t bar0 = sbase + L::kBarOff;
    auto q_full = [&](int x) { return bar0 + 8u * x; };
    auto kv_full = [&](int s) { return bar0 + 8u * (2 + s); };
    auto kv_empty = [&](int s) { return bar0 + 8u * (2 + NSTAGE + s); };
    auto s_full = [&](int x) { return bar0 + 8u * (2 + 2 * NSTAGE + x); };
    auto p_ready = [&](int x) { return bar0 + 8u * (4 + 2 * NSTAGE + x); };
    auto o_full = [&](int x) { return bar0 + 8u * (6 + 2 * NSTAGE + x); };
    volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(smem + L::kMiscOff);
    volatile int* keepflag = reinterpret_cast<volatile int*>(smem + L::kMiscOff + 4);          // [2][2]
    volatile int* votes = reinterpret_cast<volatile int*>(smem + L::kMiscOff + 4 + 16);        // [2][2][4]
    volatile float* wmax = reinterpret_cast<volatile float*>(smem + L::kMiscOff + 4 + 16 + 64);  // [2][2][4]

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int bh = blockIdx.y;
    const int tile0 = blockIdx.x * 2;
    const bool active1 = (tile0 + 1) < a.n_mma_tiles;
    const int nX = active1 ? 2 : 1;
    const int T_c = a.T_c;

    // ------------------------------------------------------------------ setup
    if (warp == kProducerWarp && lane == 0) {
        prefetch_tmap(&tm_q);
        prefetch_tmap(&tm_k);
        prefetch_tmap(&tm_v);
        for (int x = 0; x < 2; ++x) {
            mbar_init(q_full(x), 1);
            mbar_init(s_full(x), 1);
            mbar_init(p_ready(x), 128);
            mbar_init(o_full(x), 1);
        }
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(kv_full(s), 1);
            mbar_init(kv_empty(s), 1);
        }
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
        if (warp == kProducerWarp) {
        // ============================================================== TMA producer (a1)
        if (lane == 0) {
            for (int x = 0; x < nX; ++x) {
                mbar_arrive_expect_tx(q_full(x), L::kQSlotBytes);
                for (int h = 0; h < kSubD; ++h)
                    tma_load_3d(q_smem + x * L::kQSlotBytes + h * L::kSubQBytes, &tm_q, h * 64, (tile0 + x) * 128, bh,
                                q_full(x));
            }
            int stage = 0;
            uint32_t phase = 0;
            for (int e = 0; e < 2 * T_c; ++e) {       // ring entries: K_0, V_0, K_1, V_1, ...
                if (e >= NSTAGE) mbar_wait(kv_empty(stage), phase ^ 1u);
                mbar_arrive_expect_tx(kv_full(stage), L::kKVStageBytes);
                const CUtensorMap* tm = (e & 1) ? &tm_v : &tm_k;
                for (int h = 0; h < kSubD; ++h)
                    tma_load_3d(kv_smem + stage * L::kKVStageBytes + h * L::kSubKVBytes, tm, h * 64, (e >> 1) * BC, bh,
                                kv_full(stage));
                if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
            }
        }
        __syncwarp();
        } else if (warp == kMmaWarp) {
        // ============================================================== MMA issuer (a2, a6)
        if (lane == 0) {
            auto issue_qk = [&](int x, uint32_t kaddr) {
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t off = (kk >> 2) * L::kSubQBytes + (kk & 3) * 32;
                    const uint32_t koff = (kk >> 2) * L::kSubKVBytes + (kk & 3) * 32;
                    umma_ss(tmem_base + x * BC, umma_smem_desc_sw128(q_smem + x * L::kQSlotBytes + off, 16, 1024),
                            umma_smem_desc_sw128(kaddr + koff, 16, 1024), kIdescQK, kk > 0);
                }
            };
            auto issue_pv = [&](int x, uint32_t vaddr, bool acc) {
#pragma unroll
                for (int kk = 0; kk < BC / 16; ++kk) {
                    // 16 keys = 16 rows of 128 B; d sub-tiles (64 columns) are L::kSubKVBytes apart (LBO)
                    umma_ts(tmem_base + 2 * BC + x * D, tmem_base + x * BC + kk * 8,
                            umma_smem_desc_sw128(vaddr + kk * 2048, L::kSubKVBytes, 1024), kIdescPV, acc || kk > 0);
                }
            };
            int stage = 0;
            uint32_t phase = 0;
            auto advance = [&]() { if (++stage == NSTAGE) { stage = 0; phase ^= 1u; } };

            for (int x = 0; x < nX; ++x) mbar_wait(q_full(x), 0);
            mbar_wait(kv_full(stage), phase);
            tc_fence_after();
            for (int x = 0; x < nX; ++x) {
                issue_qk(x, kv_smem + stage * L::kKVStageBytes);
                umma_commit(s_full(x));
            }
            umma_commit(kv_empty(stage));
            advance();

            for (int j = 0; j < T_c; ++j) {
                const int v_stage = stage;
                const uint32_t v_phase = phase;
                advance();
                const bool has_next = (j + 1) < T_c;
                const int k_stage = stage;
                const uint32_t k_phase = phase;
                if (has_next) advance();
                bool v_waited = false, k_waited = false;
                for (int x = 0; x < nX; ++x) {
                    mbar_wait(p_ready(x), j & 1);
                    tc_fence_after();
                    const int keep = kSparse ? keepflag[x * 2 + (j & 1)] : 1;
                    if (keep) {
                        if (!v_waited) { mbar_wait(kv_full(v_stage), v_phase); tc_fence_after(); v_waited = true; }
                        issue_pv(x, kv_smem + v_stage * L::kKVStageBytes, j > 0);
                    }
                    if (has_next) {
                        if (!k_waited) { mbar_wait(kv_full(k_stage), k_phase); tc_fence_after(); k_waited = true; }
                        issue_qk(x, kv_smem + k_stage * L::kKVStageBytes);
                        umma_commit(s_full(x));
                    } else {
                        umma_commit(o_full(x));
                    }
                }
                if (!v_waited) mbar_wait(kv_full(v_stage), v_phase);
                umma_commit(kv_empty(v_stage));
                if (has_next) umma_commit(kv_empty(k_stage));
            }
        }
        __syncwarp();
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
        int n_exec = 0, n_skip = 0;

        for (int j = 0; j < T_c; ++j) {
            const int par = j & 1;
            mbar_wait(s_full(x), par);
            tc_fence_after();
            uint32_t su[BC / 32][32];                         // this thread's row of S_ij (fp32 bits)
#pragma unroll
            for (int c = 0; c < BC / 32; ++c) tmem_ld_x32(tS + c * 32, su[c]);
            tmem_wait_ld();
#define S_AT(c) __uint_as_float(su[(c) >> 5][(c) & 31])
            const int valid_cols = a.N - j * BC;             // ragged last K tile: columns beyond N are -inf
            if (valid_cols < BC) {
#pragma unroll
                for (int c = 0; c < BC; ++c)
                    if (c >= valid_cols) su[c >> 5][c & 31] = 0xff800000u;
            }
            float mx0 = S_AT(0), mx1 = S_AT(1), mx2 = S_AT(2), mx3 = S_AT(3);   // 4 independent max chains
#pragma unroll
            for (int c = 4; c < BC; c += 4) {
                mx0 = fmaxf(mx0, S_AT(c));
                mx1 = fmaxf(mx1, S_AT(c + 1));
                mx2 = fmaxf(mx2, S_AT(c + 2));
                mx3 = fmaxf(mx3, S_AT(c + 3));
            }
            const float mhat2 = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * scale_log2;   // tile-local row max (a3)

            // ---- predicate and all-rows vote (a4)
            bool skip_grp = false, keep_any = true;
            float grp_margin = INFINITY;
            if (kSparse && j > 0) {
                const float ref = (mode == kModeDynamic) ? (m_used + fast_log2(l)) : m_true;
                const float t2 = mhat2 - ref;                // Eq. 5 in log2 units
                const bool row_skip = !row_valid || (t2 < lambda_log2);
                const int wskip = __all_sync(0xffffffffu, row_skip);
                if (want_margin) {
                    float tm = row_valid ? t2 : -INFINITY;
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) tm = fmaxf(tm, __shfl_xor_sync(0xffffffffu, tm, o));
                    if (lane == 0) wmax[(x * 2 + par) * 4 + w] = tm;
                }
                if (lane == 0) votes[(x * 2 + par) * 4 + w] = wskip;
                named_bar_sync(1 + x, 128);
                const int v0 = votes[(x * 2 + par) * 4 + 0], v1 = votes[(x * 2 + par) * 4 + 1];
                const int v2 = votes[(x * 2 + par) * 4 + 2], v3 = votes[(x * 2 + par) * 4 + 3];
                if (G == 1) {
                    skip_grp = v0 && v1 && v2 && v3;
                    keep_any = !skip_grp;
                    if (want_margin)
                        grp_margin = fmaxf(fmaxf(wmax[(x * 2 + par) * 4 + 0], wmax[(x * 2 + par) * 4 + 1]),
                                           fmaxf(wmax[(x * 2 + par) * 4 + 2], wmax[(x * 2 + par) * 4 + 3]));
                } else {
                    const bool s0 = v0 && v1, s1 = v2 && v3;
                    skip_grp = grp ? s1 : s0;
                    keep_any = !(s0 && s1);
                    if (want_margin)
                        grp_margin = fmaxf(wmax[(x * 2 + par) * 4 + 2 * grp], wmax[(x * 2 + par) * 4 + 2 * grp + 1]);
                }
                if (want_margin) grp_margin = (grp_margin - lambda_log2) * kLn2;
            }
            if (grp_leader && grp_valid) {                   // a9 + optional parity outputs
                if (skip_grp) ++n_skip; else ++n_exec;
                if (kDebug) {
                    if (a.skip_mask) a.skip_mask[tile_row + j] = skip_grp ? 1 : 0;
                    if (want_margin) a.margin[tile_row + j] = grp_margin;
                }
            }

            if (kSparse && !keep_any) {                      // a7: skipped -- m, l, O untouched
                if (r == 0) keepflag[x * 2 + par] = 0;
                tc_fence_before();
                mbar_arrive(p_ready(x));
                continue;
            }

            if (kSparse && G == 2 && skip_grp) {
                // this half skipped but its partner half kept: contribute P = 0, statistics untouched
                uint32_t z[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) z[i] = 0u;
#pragma unroll
                for (int c = 0; c < BC / 32; ++c) tmem_st_x16(tS + c * 16, z);
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
                        const float p0 = fast_exp2(fmaf(__uint_as_float(su[c][2 * i]), scale_log2, neg_m));
                        const float p1 = fast_exp2(fmaf(__uint_as_float(su[c][2 * i + 1]), scale_log2, neg_m));
                        rs0 += p0;
                        rs1 += p1;
                        pk[i] = pack_bf16x2(p0, p1);
                    }
                    tmem_st_x16(tS + c * 16, pk);
                }
                l += rs0 + rs1;
            }
#undef S_AT
            tmem_wait_st();
            tc_fence_before();
            if (kSparse && r == 0) keepflag[x * 2 + par] = 1;
            mbar_arrive(p_ready(x));
        }

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
