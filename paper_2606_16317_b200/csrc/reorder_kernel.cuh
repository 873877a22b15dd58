// Token re-ordering: gather / scatter of bf16 token rows by a permutation.
//
// HBM-bound: every row (D * 2 = 128 or 256 bytes) is read once and written once, 16 bytes per thread, so a row is
// one fully coalesced 128 / 256-byte segment on both sides (only the row order differs).  The permutation
// (4 bytes per row, shared by all B*H heads) stays in L2.  Grid: a multiple of the SM count, grid-stride over rows.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dsa {

// kLanes = threads per row = D * 2 / 16.  rows = B*H*N.
template <int kLanes>
__global__ void __launch_bounds__(256)
reorder_tokens_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, const int32_t* __restrict__ perm,
                      long long rows, int N, int inverse) {
    constexpr int kRowsPerBlock = 256 / kLanes;
    const int lane = threadIdx.x % kLanes;
    const int sub = threadIdx.x / kLanes;
    constexpr int kUnroll = 4;                       // rows in flight per thread: enough loads to cover HBM latency
    const long long stride = static_cast<long long>(gridDim.x) * kRowsPerBlock * kUnroll;
    for (long long base = (static_cast<long long>(blockIdx.x) * kUnroll) * kRowsPerBlock + sub; base < rows; base += stride) {
        uint4 v[kUnroll];
        long long to[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            const long long r = base + static_cast<long long>(u) * kRowsPerBlock;
            to[u] = -1;
            if (r < rows) {
                const long long head = r / N;
                const int p = static_cast<int>(r - head * N);
                const long long other = head * N + __ldg(perm + p);
                const long long from = inverse ? r : other;
                to[u] = inverse ? other : r;
                v[u] = __ldcs(src + from * kLanes + lane);      // streamed: read once
            }
        }
#pragma unroll
        for (int u = 0; u < kUnroll; ++u)
            if (to[u] >= 0) __stcs(dst + to[u] * kLanes + lane, v[u]);
    }
}

}  // namespace dsa
