// Row-level accuracy-vs-recall analysis of PAPER.md Appendix A.1 (lines 249-275): "We sample random rows from the P
// matrix and apply Top-K with different K values to ablate the recall rate.  Excess Kurtosis is used to measure the
// 'tailedness' of a data distribution."  For each sampled query row r of head bh, over ALL N keys:
//     p = softmax(scale * q_r K^T),   kurtosis = m4 / m2^2 - 3 of the N values of p (population moments),
//     for every K of a grid: Top-K = keys with p >= the K-th largest p,  recall = sum_TopK p,
//     O' = sum_TopK p v / recall (Eq. 1's renormalised output),  MAE = mean_d |O_d - O'_d|.
// An offline analysis tool, not the hot path: one CTA of 256 threads per sampled row, the row's exponentials e = exp(s - max)
// in a global scratch line that stays in L2; the K-th largest value is found exactly by a bitwise radix select on the
// fp32 bit patterns (31 counting passes per K), with no sort.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace dsa {

constexpr int kRowCurveThreads = 256;

__device__ __forceinline__ double block_sum_f64(double v, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();                                          // red may still be read from the previous call
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int i = 0; i < kRowCurveThreads / 32; ++i) t += red[i];
    return t;
}

__device__ __forceinline__ float block_max_f32(float v, float* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    float t = red[0];
#pragma unroll
    for (int i = 1; i < kRowCurveThreads / 32; ++i) t = fmaxf(t, red[i]);
    return t;
}

// D / 32 consecutive elements of a bf16 row per lane -> fp32
template <int D>
__device__ __forceinline__ void load_row_slice(const __nv_bfloat16* row, int lane, float (&x)[D / 32]) {
    if constexpr (D == 128) {
        const uint2 u = *reinterpret_cast<const uint2*>(row + lane * 4);
        const float2 a = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&u.x));
        const float2 b = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&u.y));
        x[0] = a.x; x[1] = a.y; x[2] = b.x; x[3] = b.y;
    } else {
        const float2 a = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(row + lane * 2));
        x[0] = a.x; x[1] = a.y;
    }
}

// rows: [n_rows][2] int32 = (bh, r);  keep: [n_K] int32, 1 <= K <= N;  scratch: [n_rows][N] fp32
// kurt_out: [n_rows] fp64;  recall_out, mae_out: [n_rows][n_K] fp64
template <int D>
__global__ void __launch_bounds__(kRowCurveThreads)
row_topk_curve_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ k,
                      const __nv_bfloat16* __restrict__ v, int N, float scale, const int32_t* __restrict__ rows,
                      const int32_t* __restrict__ keep, int n_K, float* __restrict__ scratch,
                      double* __restrict__ kurt_out, double* __restrict__ recall_out, double* __restrict__ mae_out) {
    constexpr int E = D / 32;                                // elements of a row per lane
    constexpr int kWarps = kRowCurveThreads / 32;
    __shared__ double red64[kWarps];
    __shared__ float red32[kWarps];
    __shared__ float osum[kWarps][D];
    __shared__ float o_dense[D];
    __shared__ int count;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int bh = rows[2 * blockIdx.x], r = rows[2 * blockIdx.x + 1];
    const __nv_bfloat16* kb = k + static_cast<size_t>(bh) * N * D;
    const __nv_bfloat16* vb = v + static_cast<size_t>(bh) * N * D;
    float* e = scratch + static_cast<size_t>(blockIdx.x) * N;

    // ---- logits s_c = scale * <q_r, k_c> (one key per warp step), row max
    float qx[E];
    load_row_slice<D>(q + (static_cast<size_t>(bh) * N + r) * D, lane, qx);
    float mx = -INFINITY;
    for (int c = warp; c < N; c += kWarps) {
        float kx[E];
        load_row_slice<D>(kb + static_cast<size_t>(c) * D, lane, kx);
        float d = 0.f;
#pragma unroll
        for (int i = 0; i < E; ++i) d = fmaf(qx[i], kx[i], d);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
        d *= scale;
        if (lane == 0) e[c] = d;
        mx = fmaxf(mx, d);
    }
    mx = block_max_f32(mx, red32);                            // (its barriers also publish the logits to the CTA)

    // ---- e_c = exp(s_c - max), their sum
    double part = 0.0;
    for (int c = threadIdx.x; c < N; c += kRowCurveThreads) {
        const float ec = expf(e[c] - mx);
        e[c] = ec;
        part += static_cast<double>(ec);
    }
    const double total = block_sum_f64(part, red64);
    const double inv_total = 1.0 / total;

    // ---- excess kurtosis of p = e / total: population moments about the mean 1 / N
    const double mean = 1.0 / static_cast<double>(N);
    double s2 = 0.0, s4 = 0.0;
    for (int c = threadIdx.x; c < N; c += kRowCurveThreads) {
        const double d = static_cast<double>(e[c]) * inv_total - mean;
        const double d2 = d * d;
        s2 += d2;
        s4 += d2 * d2;
    }
    const double m2 = block_sum_f64(s2, red64) / static_cast<double>(N);
    const double m4 = block_sum_f64(s4, red64) / static_cast<double>(N);
    if (threadIdx.x == 0) kurt_out[blockIdx.x] = m4 / (m2 * m2) - 3.0;      // (a constant row: 0 / 0 = NaN, as the oracle)

    // sum over the keys with e_c >= thr of e_c v_c (per dimension, fp32) and of e_c (fp64): every warp takes 32 keys at a
    // time, ballots the retained ones and walks the set bits, so that discarded keys cost no V traffic
    auto weighted_sum = [&](float thr, float* o_final, double* mass_final) {
        float acc[E];
#pragma unroll
        for (int i = 0; i < E; ++i) acc[i] = 0.f;
        double mass = 0.0;
        for (int c0 = warp * 32; c0 < N; c0 += kWarps * 32) {
            const int c = c0 + lane;
            const float ec = c < N ? e[c] : -1.f;
            uint32_t m = __ballot_sync(0xffffffffu, ec >= thr);
            if (ec >= thr) mass += static_cast<double>(ec);
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1;
                const float w = __shfl_sync(0xffffffffu, ec, b);
                float vx[E];
                load_row_slice<D>(vb + static_cast<size_t>(c0 + b) * D, lane, vx);
#pragma unroll
                for (int i = 0; i < E; ++i) acc[i] = fmaf(w, vx[i], acc[i]);
            }
        }
        __syncthreads();                                      // osum may still be read from the previous call
#pragma unroll
        for (int i = 0; i < E; ++i) osum[warp][lane * E + i] = acc[i];
        const double tot = block_sum_f64(mass, red64);        // (barriers inside)
        if (threadIdx.x < D) {
            float t = 0.f;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) t += osum[w][threadIdx.x];
            o_final[threadIdx.x] = t;
        }
        __syncthreads();
        *mass_final = tot;
    };

    // ---- dense output O = sum_c p_c v_c
    __shared__ float o_kept[D];
    double mass_all;
    weighted_sum(0.f, o_dense, &mass_all);

    // ---- for every K: the K-th largest e (bitwise radix select), recall, O', MAE
    for (int ik = 0; ik < n_K; ++ik) {
        const int K = keep[ik];
        uint32_t prefix = 0u;
        int remaining = K;
        for (int bit = 30; bit >= 0; --bit) {                 // e in (0, 1]: the sign bit is clear
            const uint32_t cand = (prefix | (1u << bit)) >> bit;
            int cnt = 0;
            for (int c = threadIdx.x; c < N; c += kRowCurveThreads) cnt += ((__float_as_uint(e[c]) >> bit) == cand) ? 1 : 0;
            cnt = __reduce_add_sync(0xffffffffu, cnt);
            if (threadIdx.x == 0) count = 0;
            __syncthreads();
            if (lane == 0) atomicAdd(&count, cnt);
            __syncthreads();
            const int n_set = count;                          // keys that share the prefix and have this bit set
            __syncthreads();
            if (n_set >= remaining) prefix |= 1u << bit;      // the K-th largest is among them
            else remaining -= n_set;
        }
        const float thr = __uint_as_float(prefix);
        double mass_kept;
        weighted_sum(thr, o_kept, &mass_kept);
        double err = 0.0;
        if (threadIdx.x < D)
            err = fabs(static_cast<double>(o_dense[threadIdx.x]) * inv_total -
                       static_cast<double>(o_kept[threadIdx.x]) / mass_kept);
        const double err_sum = block_sum_f64(err, red64);
        if (threadIdx.x == 0) {
            recall_out[static_cast<size_t>(blockIdx.x) * n_K + ik] = mass_kept * inv_total;
            mae_out[static_cast<size_t>(blockIdx.x) * n_K + ik] = err_sum / static_cast<double>(D);
        }
    }
}

}  // namespace dsa
