// Device helpers of the epoch-boundary segmenter (a1), shared by segmenter.cu and by the K = 4 chain kernel, which segments its
// own branch inline (same expressions, same bits) so that the segmenter kernels can run beside it instead of before it.
#pragma once
#include "epx_internal.h"

namespace epxseg {

__device__ __forceinline__ int count_less(const double* __restrict__ tau, int n, double h, bool or_equal)
{
    int lo = 0, hi = n;   // first index whose tau is NOT (< h) / (<= h)
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        double t = tau[mid];
        bool in = or_equal ? (t <= h) : (t < h);
        if (in) lo = mid + 1; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ void branch_ends(int b, const int32_t* __restrict__ parent, const double* __restrict__ height,
                                            const double* __restrict__ child_h, const double* __restrict__ parent_h,
                                            double& hc, double& hp)
{
    if (parent) {
        hc = height[b];
        int p = parent[b];
        hp = p < 0 ? hc : height[p];
    } else {
        hc = child_h[b];
        hp = parent_h[b];
    }
}

}  // namespace epxseg
