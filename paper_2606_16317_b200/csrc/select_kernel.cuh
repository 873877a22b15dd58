// Block selectors on the block-mass matrix (Table 1 / Fig. 3 comparison methods): Top-K keeps a fixed
// number of tiles per row of tiles, Top-P keeps tiles in order of decreasing mass until their share reaches P.
// One CTA per row of tiles; every thread ranks its tiles against the whole row held in shared memory (O(T_c^2) per
// row: T_c is a few hundred, the whole matrix a few MB -- an offline analysis step, not a hot path).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dsa {

constexpr int kSelectMaxTc = 4096;

// kind 0: Top-K, keep the n_keep tiles of largest mass.  kind 1: Top-P, keep a tile iff the mass of the tiles ahead of
// it (larger mass; equal mass and lower index) is < p * row total.  Tile 0 is always kept.  skip_out: 1 = skip.
__global__ void __launch_bounds__(256)
select_blocks_kernel(const float* __restrict__ mass, uint8_t* __restrict__ skip_out, int T_c, int kind, int n_keep, double p) {
    extern __shared__ float row[];
    const size_t base = (static_cast<size_t>(blockIdx.y) * gridDim.x + blockIdx.x) * static_cast<size_t>(T_c);
    for (int j = threadIdx.x; j < T_c; j += blockDim.x) row[j] = mass[base + j];
    __syncthreads();
    double total = 0.0;
    if (kind == 1)
        for (int j = 0; j < T_c; ++j) total += static_cast<double>(row[j]);   // same order in every thread
    for (int j = threadIdx.x; j < T_c; j += blockDim.x) {
        const float mj = row[j];
        int ahead = 0;
        double ahead_mass = 0.0;
        for (int i = 0; i < T_c; ++i) {
            const float mi = row[i];
            if (mi > mj || (mi == mj && i < j)) {
                ++ahead;
                ahead_mass += static_cast<double>(mi);
            }
        }
        const bool keep = (j == 0) || (kind == 0 ? ahead < n_keep : ahead_mass < p * total);
        skip_out[base + j] = keep ? 0 : 1;
    }
}

// The "ideal" mask of PAPER.md section 3 (lines 105-109) at block level: per row of tiles, tiles are moved from the kept
// set K to the discarded set S in order of increasing mass while the variance bound of Eq. 3 holds,
//     sum_S q_j + (S_1 / (1 - S_1))^2 sum_K q_j <= Theta,     S_1 = sum_S P_j,
// with P_j / q_j the block sums of p / p^2 averaged over the rows of the Q tile (R14).  The scan stops at the
// first tile whose removal would violate the bound.  Tile 0 is never a candidate (MASK mode keeps it regardless).
// One CTA per row of tiles; thread j ranks tile j against the whole row (ascending mass, ties by lower index).
__global__ void __launch_bounds__(256)
select_blocks_greedy_kernel(const float* __restrict__ mass, const float* __restrict__ sqmass, uint8_t* __restrict__ skip_out,
                            int T_c, int N, int tile_q, double theta) {
    extern __shared__ float rowbuf[];
    float* row = rowbuf;
    float* rsq = rowbuf + T_c;
    // rank of the first tile whose removal would violate Eq. 3; it lives in the rank slot of tile 0, which is never a
    // candidate, so that the kernel's shared memory is exactly 3 T_c floats (48 KB at T_c = kSelectMaxTc, the default limit)
    int& first_violation = *reinterpret_cast<int*>(rowbuf + 2 * T_c);
    const size_t base = (static_cast<size_t>(blockIdx.y) * gridDim.x + blockIdx.x) * static_cast<size_t>(T_c);
    for (int j = threadIdx.x; j < T_c; j += blockDim.x) { row[j] = mass[base + j]; rsq[j] = sqmass[base + j]; }
    if (threadIdx.x == 0) first_violation = T_c;
    __syncthreads();
    const int rows = min(tile_q, N - static_cast<int>(blockIdx.x) * tile_q);
    const double inv_rows = 1.0 / static_cast<double>(rows);
    double total_sq = 0.0;
    for (int j = 0; j < T_c; ++j) total_sq += static_cast<double>(rsq[j]);     // same order in every thread
    for (int j = threadIdx.x; j < T_c; j += blockDim.x) {
        if (j == 0) continue;
        const float mj = row[j];
        int rank = 0;
        double s_mass = static_cast<double>(mj), s_sq = static_cast<double>(rsq[j]);   // S = this tile and every tile before it
        for (int i = 1; i < T_c; ++i) {
            const float mi = row[i];
            if (mi < mj || (mi == mj && i < j)) {
                ++rank;
                s_mass += static_cast<double>(mi);
                s_sq += static_cast<double>(rsq[i]);
            }
        }
        const double s1 = s_mass * inv_rows;
        const double ratio = s1 / (1.0 - s1);
        const double lhs = s_sq * inv_rows + ratio * ratio * ((total_sq - s_sq) * inv_rows);
        if (!(s1 < 1.0) || !(lhs <= theta)) atomicMin(&first_violation, rank);
        rowbuf[2 * T_c + j] = __int_as_float(rank);
    }
    __syncthreads();
    for (int j = threadIdx.x; j < T_c; j += blockDim.x)
        skip_out[base + j] = (j > 0 && __float_as_int(rowbuf[2 * T_c + j]) < first_violation) ? 1 : 0;
}

}  // namespace dsa
