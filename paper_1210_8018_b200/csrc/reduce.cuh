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
#ifdef LGF_REDUCE_SKIP   /* timing-only probe: no final sum (F, theta and the stop decision are NOT produced) */
    if (last && threadIdx.x == 0) ctrl->iter += count_iter ? 1 : 0;
    return;
#endif
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

// The same in two levels, for the kernel of the inner loop.  In finish_measure ONE block adds the partial sums of the
// whole grid while the rest of the GPU idles: 5.8 us of the 200 us of the link kernel at 32^4 (8192 blocks), 82 us at
// 64^4 (131072 blocks; timing probe -DLGF_REDUCE_SKIP, profiles/r02_reduce.md).  Here the blocks form groups of
// LGF_REDUCE_GROUP consecutive indices; the last block of a GROUP to arrive adds the group's partial sums (while other
// groups are still at work), the last GROUP to finish adds the group sums.  Every sum runs over fixed indices in a
// fixed order, so F and theta are bitwise reproducible whichever blocks happen to be last; they differ from the
// one-level sums in the order of the additions only.
// Scratch: `partials` holds the G block partials as before; `gred` is a region of its own (the one-level kernels,
// whose grids differ, never write it): NG group partials (pairs of doubles) followed by NG unsigned group tickets,
// NG = ceil(G / LGF_REDUCE_GROUP).  The tickets start at zero (lgf_bind clears the region) and wrap back to zero
// with the last arrival of every launch.  reduce2l_bytes(G) is what the region must hold for grids up to G blocks.
#ifndef LGF_REDUCE_GROUP
#define LGF_REDUCE_GROUP 64
#endif
__host__ __device__ inline size_t reduce2l_bytes(int64_t max_blocks)
{
    const size_t ng = (size_t)((max_blocks + LGF_REDUCE_GROUP - 1) / LGF_REDUCE_GROUP) + 1;
    return ng * (sizeof(double2) + sizeof(unsigned)) + 16;
}
template <int THREADS>
__device__ __forceinline__ void finish_measure_2l(double trF, double th, int64_t V, Ctrl *ctrl, double *partials, void *gred,
                                                  double2 *hist, double eps, int count_iter)
{
    static_assert(LGF_REDUCE_GROUP <= THREADS, "a group is summed by one pass of the block");
    block_sum2<THREADS>(trF, th);
    __shared__ int role;                                   // 0: done, 1: last block of its group, 2: last group
    const unsigned G = gridDim.x, GS = LGF_REDUCE_GROUP, NG = (G + GS - 1) / GS;
    double2 *bpart = (double2 *)partials, *gpart = (double2 *)gred;
    unsigned *gtick = (unsigned *)(gpart + NG);
    const unsigned grp = blockIdx.x / GS;
    const unsigned gsize = (grp + 1) * GS <= G ? GS : G - grp * GS;
    if (threadIdx.x == 0) {
        bpart[blockIdx.x] = make_double2(trF, th);
        __threadfence();
        const unsigned tk = atomicInc(&gtick[grp], gsize - 1);
        role = (tk == gsize - 1) ? 1 : 0;
    }
    __syncthreads();
    if (!role) return;
    __threadfence();
    double f = 0, t = 0;
    if (threadIdx.x < gsize) {
        const double2 v = __ldcg(bpart + (size_t)grp * GS + threadIdx.x);
        f = v.x; t = v.y;
    }
    block_sum2<THREADS>(f, t);
    if (threadIdx.x == 0) {
        gpart[grp] = make_double2(f, t);
        __threadfence();
        const unsigned tk = atomicInc(&ctrl->ticket, NG - 1);
        role = (tk == NG - 1) ? 2 : 0;
    }
    __syncthreads();
    if (role != 2) return;
    __threadfence();
    f = 0; t = 0;
    for (unsigned i = threadIdx.x; i < NG; i += THREADS) {
        const double2 v = __ldcg(gpart + i);
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
