// reduce.cuh -- fixed-order FP64 reductions of F (eq. 1.1) and theta (eq. 1.4,
// PAPER.md:59) shared by the kernels that measure (CUDA path only).
#pragma once
#include "common.cuh"

#ifndef LGF_REDUCE_UNROLL
#define LGF_REDUCE_UNROLL 8   /* 1: the plain loop (same sums; tuning A/B, profiles/r02_link_kernel.md) */
#endif

namespace lgf {

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum of (a, b) over the block; result valid in thread 0.  Order is fixed by the code, so
// the sums are bitwise reproducible run to run.
template <int THREADS> __device__ __forceinline__ void block_sum2(double &a, double &b)
{
    __shared__ double sa[THREADS / 32], sb[THREADS / 32];
    a = warp_sum(a); b = warp_sum(b);
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { sa[w] = a; sb[w] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double ta = 0, tb = 0;
#pragma unroll
        for (int i = 0; i < THREADS / 32; i++) { ta += sa[i]; tb += sb[i]; }
        a = ta; b = tb;
    }
    __syncthreads();
}

// Block partials -> F, theta.  Every block writes its pair of partial sums; the last block to
// arrive (ticket counter) adds all partials in index order, so the result does not depend on
// the order in which blocks ran.  It also takes the stop decision of Alg. 1 line 2
// (theta <= eps; reading R2) and appends (F, theta) to the history.
// Must be called by every thread of every block of the grid.
template <int THREADS>
__device__ __forceinline__ void finish_measure(double trF, double th, int64_t V, Ctrl *ctrl, double *partials,
                                               double2 *hist, double eps, int count_iter)
{
    block_sum2<THREADS>(trF, th);
    __shared__ bool last;
    if (threadIdx.x == 0) {
        partials[2 * (int64_t)blockIdx.x] = trF;
        partials[2 * (int64_t)blockIdx.x + 1] = th;
        __threadfence();
        const unsigned tk = atomicInc(&ctrl->ticket, gridDim.x - 1); // wraps back to 0 for the next launch
        last = (tk == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    // One CTA adds gridDim.x pairs while the rest of the GPU idles (8192 pairs at 32^4, 131072 at 64^4), so the
    // loads are issued eight at a time per thread, as 16-byte pairs; the additions keep the index order
    // i, i + THREADS, i + 2 THREADS, ... of each thread, i.e. the result is bitwise that of the plain loop.
    double f = 0, t = 0;
    const double2 *pp = (const double2 *)partials;
    constexpr int UNR = LGF_REDUCE_UNROLL;
    unsigned i = threadIdx.x;
    for (; i + (UNR - 1) * THREADS < gridDim.x; i += UNR * THREADS) {
        double2 v[UNR];
#pragma unroll
        for (int u = 0; u < UNR; u++) v[u] = __ldcg(pp + i + u * THREADS);
#pragma unroll
        for (int u = 0; u < UNR; u++) { f += v[u].x; t += v[u].y; }
    }
    for (; i < gridDim.x; i += THREADS) {
        const double2 v = __ldcg(pp + i);
        f += v.x; t += v.y;
    }
    block_sum2<THREADS>(f, t);
    if (threadIdx.x == 0) {
        const double F = f / (12.0 * (double)V), theta = t / (3.0 * (double)V);
        long long it = ctrl->iter + (count_iter ? 1 : 0);
        ctrl->F = F; ctrl->theta = theta; ctrl->iter = it;
        if (it < LGF_HIST_CAP) hist[it] = make_double2(F, theta);
        if (!(theta == theta) || theta > 1.0e300) ctrl->done = 2;
        else if (theta <= eps) ctrl->done = 1;
    }
}

} // namespace lgf
