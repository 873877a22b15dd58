// Quality statistics of a sparse run against the dense run of the same inputs, computed on the device so that the
// harness never touches the values with anything but this library:
//   recall_r = e^{lse_retained_r - lse_dense_r}: the share of row r's softmax mass the retained tiles hold
//               -> minimum and sum over rows
//   |O' - O|: element-wise error of the sparse output against the dense one -> maximum and sum
// Grid-stride reductions (HBM-bound, a few MB): warp shuffle, one atomic per warp.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace dsa {

__global__ void stats_init_kernel(double* out, double v0, double v1) {
    out[0] = v0;
    out[1] = v1;
}

// positive doubles order like their bit patterns: atomicMin / atomicMax on the 64-bit integer view.
// In the minimum a NaN beats everything (a broken run must not report a healthy minimum): positive doubles also order
// like SIGNED 64-bit integers, and a NaN with its sign bit set is below all of them
__device__ __forceinline__ void atomic_min_pos_or_nan(double* addr, double v) {
    const long long bits = (v != v) ? static_cast<long long>(0xfff8000000000000ull) : __double_as_longlong(v);
    atomicMin(reinterpret_cast<long long*>(addr), bits);
}
__device__ __forceinline__ double min_or_nan(double a, double b) { return (a != a || b != b) ? NAN : fmin(a, b); }
__device__ __forceinline__ void atomic_max_pos(double* addr, double v) {
    atomicMax(reinterpret_cast<unsigned long long*>(addr), static_cast<unsigned long long>(__double_as_longlong(v)));
}

// out[0] = min_r recall_r (NaN if any row's recall is NaN), out[1] = sum_r recall_r   (out pre-set to {+inf, 0})
__global__ void __launch_bounds__(256)
recall_stats_kernel(const float* __restrict__ lse_retained, const float* __restrict__ lse_dense, long long n, double* out) {
    double mn = INFINITY, sm = 0.0;
    for (long long i = blockIdx.x * 256ll + threadIdx.x; i < n; i += static_cast<long long>(gridDim.x) * 256) {
        const double rec = exp(static_cast<double>(lse_retained[i]) - static_cast<double>(lse_dense[i]));
        mn = min_or_nan(mn, rec);
        sm += rec;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mn = min_or_nan(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        sm += __shfl_xor_sync(0xffffffffu, sm, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomic_min_pos_or_nan(out, mn);
        atomicAdd(out + 1, sm);
    }
}

// out[0] = max |a - b|, out[1] = sum |a - b| over n bf16 elements (n even; out pre-set to {0, 0})
__global__ void __launch_bounds__(256)
output_error_kernel(const __nv_bfloat162* __restrict__ a, const __nv_bfloat162* __restrict__ b, long long n2, double* out) {
    float mx = 0.f;
    double sm = 0.0;
    for (long long i = blockIdx.x * 256ll + threadIdx.x; i < n2; i += static_cast<long long>(gridDim.x) * 256) {
        const float2 x = __bfloat1622float2(a[i]), y = __bfloat1622float2(b[i]);
        const float d0 = fabsf(x.x - y.x), d1 = fabsf(x.y - y.y);
        mx = fmaxf(mx, fmaxf(d0, d1));
        sm += static_cast<double>(d0) + static_cast<double>(d1);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        sm += __shfl_xor_sync(0xffffffffu, sm, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomic_max_pos(out, static_cast<double>(mx));
        atomicAdd(out + 1, sm);
    }
}

}  // namespace dsa
