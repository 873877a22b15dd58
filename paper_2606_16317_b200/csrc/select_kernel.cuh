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

}  // namespace dsa
