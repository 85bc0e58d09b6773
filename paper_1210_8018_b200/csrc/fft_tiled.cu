// fft_tiled.cu -- the Fourier acceleration of Algorithm 1 (lines 3-8) as a
// hand-written batched 4D FFT in three passes over HBM:
//   pass 0  (x,y) forward               one (field, z, t) plane per thread group
//   pass 1  (z,t) forward, times p_max^2/(p^2 V) (eq. 1.2; zero mode -> 0), (z,t) inverse
//           one (field, y, chunk of C consecutive x) tile per thread group, visited once
//   pass 2  (x,y) inverse
// The paper runs CUFFT as 2D+2D with a reorder kernel and a separate mask kernel
// (four passes per direction change); here the reorder is tile
// addressing and the mask and 1/V ride on the middle pass.
//
// Every 1D transform is done on a whole line held in registers -- by ONE thread for short
// lines, by TWO threads (lanes l and l^16, half a line each, one shuffle exchange) for 48 and
// 64, where a line would not fit the register file, and for 32 in FP64 square tiles, where
// halving the registers doubles the warps per tile (split_min below) -- as a fully
// unrolled decimation-in-frequency network (natural order in, digit-reversed slots out)
// with compile-time twiddles; the inverse right after the mask is the transposed
// (decimation-in-time) network, which takes digit-reversed slots and returns natural order,
// so no permutation is ever executed: slot -> frequency is a compile-time index used for
// addressing and for the mask.  Lines along the second axis of a tile go through shared
// memory (padded rows, conflict-free for 16-byte accesses); the first axis of a pass is
// loaded straight from global memory into registers and the last one stored straight back.
#ifndef LGF_F32X2
#define LGF_F32X2 1   /* packed FP32 complex arithmetic (common.cuh) for the (x,y) passes: measured faster here only */
#endif
#include "fft_lines.cuh"
#include "su3.cuh"
#include <cooperative_groups.h>

namespace lgf {

// ---------------------------------------------------------------- pass 0 / pass 2: (x,y) planes
// INVERSE = 0: load columns (lines along y) straight from global, Dif along y, through shared
//              memory, Dif along x, back through shared memory, coalesced store.
// INVERSE = 1: coalesced load into shared memory, Dif(+) along x, shared, Dif(+) along y,
//              store straight from registers.  Natural order in global memory in both cases.
template <typename T, int NA, int NB> struct XYCfg {
    typedef Tile<NA, NB, 1, split_min<T>(NA, NB)> TL;
    static constexpr int TP = TL::THREADS;             // threads of one plane
    static constexpr int CTA = cta_threads(TP);
    static constexpr int G = CTA / TP;                 // planes per CTA
    static constexpr size_t SMEM = (size_t)G * TL::ELEMS * sizeof(cx<T>);
};

// AX = 0: both axes (the pass of the 3- and 4-pass structures).  AX = 1 / 2: the x-lines / y-lines alone, the
// 1D passes of the 4 x 1D structure of the paper's comparison (LGF_OPT_FFT_PASSES = 8).
#ifndef LGF_XY_MINB
#define LGF_XY_MINB 1   /* minimum CTAs per SM asked of the (x,y) passes (register cap); tuning macro */
#endif
template <typename T, int NA, int NB, int INVERSE, int AX = 0>
__global__ void __launch_bounds__((XYCfg<T, NA, NB>::CTA), LGF_XY_MINB)
k_fft_xy(cx<T> *__restrict__ w, int64_t nplanes, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    typedef XYCfg<T, NA, NB> CF;
    typedef typename CF::TL TL;
    typedef Line<T, NA, TL::SA> LA;
    typedef Line<T, NB, TL::SB> LB;
    constexpr int TP = CF::TP, G = CF::G;
    constexpr int SIGN = INVERSE ? +1 : -1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int grp = threadIdx.x / TP, t = threadIdx.x % TP;
    cx<T> *sm = (cx<T> *)smem_raw + (size_t)grp * TL::ELEMS;
    const int64_t plane = (int64_t)blockIdx.x * G + grp;
    const bool ok = plane < nplanes && grp < G;
    cx<T> *f = w + plane * (int64_t)(NA * NB);
    int xa, ha, yb, hb;                                   // thread as (x, half) of a y-line / (ky, half) of an x-line
    line_of_thread<TL::SB>(t, xa, ha);
    line_of_thread<TL::SA>(t, yb, hb);
    const bool on_y = ok && xa < NA && t < TL::SB * NA, on_x = ok && yb < NB && t < TL::SA * NB;
    const unsigned my = __ballot_sync(0xffffffffu, on_y), mx = __ballot_sync(0xffffffffu, on_x);

    if (AX == 2) {                                        // y-lines only: global -> registers -> global, in place
        if (on_y) {
            cx<T> v[LB::NL];
#pragma unroll
            for (int i = 0; i < LB::NL; i++) v[i] = f[LB::nat(i, ha) * NA + xa];
            LB::template dif<SIGN>(v, ha, my);
#pragma unroll
            for (int q = 0; q < LB::NL; q++) f[LB::slot(q, ha) * NA + xa] = v[q];
        }
        return;
    }
    if (AX == 1) {                                        // x-lines only: contiguous lines go through shared memory
        if (ok) {
#pragma unroll
            for (int k = 0; k < (NA * NB + TP - 1) / TP; k++) {
                const int e = t + k * TP;
                if (e < NA * NB) sm[(e / NA) * TL::RS + (e % NA)] = f[e];
            }
        }
        __syncthreads();
        if (on_x) {
            cx<T> v[LA::NL];
#pragma unroll
            for (int i = 0; i < LA::NL; i++) v[i] = sm[yb * TL::RS + LA::nat(i, hb)];
            LA::template dif<SIGN>(v, hb, mx);
#pragma unroll
            for (int q = 0; q < LA::NL; q++) sm[yb * TL::RS + LA::slot(q, hb)] = v[q];
        }
        __syncthreads();
        if (ok) {
#pragma unroll
            for (int k = 0; k < (NA * NB + TP - 1) / TP; k++) {
                const int e = t + k * TP;
                if (e < NA * NB) f[e] = sm[(e / NA) * TL::RS + (e % NA)];
            }
        }
        return;
    }
    if (!INVERSE) {
        if (on_y) {                                       // line along y at x = xa
            cx<T> v[LB::NL];
#pragma unroll
            for (int i = 0; i < LB::NL; i++) v[i] = f[LB::nat(i, ha) * NA + xa];
            LB::template dif<SIGN>(v, ha, my);
#pragma unroll
            for (int q = 0; q < LB::NL; q++) sm[LB::slot(q, ha) * TL::RS + xa] = v[q];
        }
        __syncthreads();
        if (on_x) {                                       // line along x at ky = yb
            cx<T> v[LA::NL];
#pragma unroll
            for (int i = 0; i < LA::NL; i++) v[i] = sm[yb * TL::RS + LA::nat(i, hb)];
            LA::template dif<SIGN>(v, hb, mx);
#pragma unroll
            for (int q = 0; q < LA::NL; q++) sm[yb * TL::RS + LA::slot(q, hb)] = v[q];
        }
        __syncthreads();
        if (ok) {
#pragma unroll
            for (int k = 0; k < (NA * NB + TP - 1) / TP; k++) {
                const int e = t + k * TP;
                if (e < NA * NB) f[e] = sm[(e / NA) * TL::RS + (e % NA)];
            }
        }
    } else {
        if (ok) {
#pragma unroll
            for (int k = 0; k < (NA * NB + TP - 1) / TP; k++) {
                const int e = t + k * TP;
                if (e < NA * NB) sm[(e / NA) * TL::RS + (e % NA)] = f[e];
            }
        }
        __syncthreads();
        if (on_x) {
            cx<T> v[LA::NL];
#pragma unroll
            for (int i = 0; i < LA::NL; i++) v[i] = sm[yb * TL::RS + LA::nat(i, hb)];
            LA::template dif<SIGN>(v, hb, mx);
#pragma unroll
            for (int q = 0; q < LA::NL; q++) sm[yb * TL::RS + LA::slot(q, hb)] = v[q];
        }
        __syncthreads();
        if (on_y) {
            cx<T> v[LB::NL];
#pragma unroll
            for (int i = 0; i < LB::NL; i++) v[i] = sm[LB::nat(i, ha) * TL::RS + xa];
            LB::template dif<SIGN>(v, ha, my);
#pragma unroll
            for (int q = 0; q < LB::NL; q++) f[LB::slot(q, ha) * NA + xa] = v[q];
        }
    }
}

// ---------------------------------------------------------------- pass 2 with the g build fused
// (x,y) inverse of all four packed fields of one (z,t) plane in one CTA, then
// g(x) = reunit(1 + (alpha/2) w(x)) (Alg. 1 lines 9-11) straight from shared
// memory: w never goes back to HBM, rows 0, 1 of g (12 reals) do.  The fused link kernel
// (kernels_fused.cu) then reads g at x and its 8 neighbours instead of rebuilding it 9 times.
template <typename T, int NA, int NB> struct XYGCfg {
    typedef Tile<NA, NB, 1, split_min<T>(NA, NB)> TL;
    // threads of one field of one plane; whole warps when lines are split (the halves shuffle)
    static constexpr int TP = (TL::SA > 1 || TL::SB > 1) ? (TL::THREADS + 31) / 32 * 32 : TL::THREADS;
    static constexpr int TG = 4 * TP;                         // threads of one plane
    static constexpr int CTA = cta_threads(TG);
    static constexpr int G = CTA / TG;
    static constexpr size_t SMEM = (size_t)G * 4 * TL::ELEMS * sizeof(cx<T>);
    static constexpr bool FITS = SMEM <= 227 * 1024 && CTA <= 1024;
};

// g -> the g buffer, or (ACC, LGF_OPT_ACCUM_G) the accumulated transformation G(x) <- g(x) G(x):
// rows 0, 1 of G are read (Gold, loaded by the caller ahead of time), row 2 rebuilt, rows 0, 1 of
// the product Gram-Schmidt cleaned and stored.
template <typename T, bool ACC>
__device__ __forceinline__ void emit_g(cx<T> (&g)[9], const cx<T> (&Gold)[6], cx<T> *__restrict__ dst, int64_t V)
{
    if (ACC) {
        cx<T> G[9], n[9];
#pragma unroll
        for (int k = 0; k < 6; k++) G[k] = Gold[k];
        su3_row2(G);
        mul_rows<2>(g, G, n);
        reunit01<T>(n);
#pragma unroll
        for (int k = 0; k < 6; k++) dst[(int64_t)k * V] = n[k];
    } else {
#pragma unroll
        for (int k = 0; k < 6; k++) dst[(int64_t)k * V] = g[k];
    }
}
// Sites of the epilogue handled per loop trip: with ACC the loads of G for all of them are issued
// before the first product, so that the trip pays one memory latency instead of EPI_BATCH.
// 2: measured best with split 32-point lines (122 registers, two 256-thread CTAs per SM; 4 needs 160
// registers and leaves one CTA per SM: 70 instead of 56 us at 32^4, profiles/r01e_final.md).
#ifndef LGF_EPI_BATCH
#define LGF_EPI_BATCH 2
#endif
#ifndef LGF_EPI_ALL
#define LGF_EPI_ALL 0   /* 1: unroll the epilogue by LGF_EPI_BATCH without ACCUM_G too (measured: no gain) */
#endif

template <typename T, int NA, int NB, bool ACC>
__global__ void __launch_bounds__((XYGCfg<T, NA, NB>::CTA))
k_fft_xy_inv_g(const cx<T> *__restrict__ w, cx<T> *__restrict__ gbuf, int64_t V, int64_t nplanes, T a, int gexp, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    typedef XYGCfg<T, NA, NB> CF;
    typedef typename CF::TL TL;
    typedef Line<T, NA, TL::SA> LA;
    typedef Line<T, NB, TL::SB> LB;
    constexpr int TP = CF::TP, TG = CF::TG, G = CF::G;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int grp = threadIdx.x / TG, t = threadIdx.x % TG;
    const int fld = t / TP, l = t % TP;
    cx<T> *smp = (cx<T> *)smem_raw + (size_t)grp * 4 * TL::ELEMS;   // the 4 fields of this plane
    cx<T> *sm = smp + (size_t)fld * TL::ELEMS;
    const int64_t plane = (int64_t)blockIdx.x * G + grp;
    const bool ok = plane < nplanes && grp < G;
    const int64_t base = plane * (int64_t)(NA * NB);
    int xa, ha, yb, hb;
    line_of_thread<TL::SB>(l, xa, ha);
    line_of_thread<TL::SA>(l, yb, hb);
    const bool on_y = ok && xa < NA && l < TL::SB * NA, on_x = ok && yb < NB && l < TL::SA * NB;
    const unsigned my = __ballot_sync(0xffffffffu, on_y), mx = __ballot_sync(0xffffffffu, on_x);

    if (ACC && ok) {
        // the epilogue reads rows 0, 1 of G of this plane: ask L2 for them now, behind the transforms
        constexpr int LINES = (int)((size_t)NA * NB * sizeof(cx<T>) / 128);
        for (int i = t; i < 6 * LINES; i += TG) {
            const char *p = (const char *)(gbuf + (int64_t)(i / LINES) * V + base) + (size_t)(i % LINES) * 128;
            asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
        }
    }
    if (ok) {
        const cx<T> *f = w + (int64_t)fld * V + base;
#pragma unroll
        for (int k = 0; k < (NA * NB + TP - 1) / TP; k++) {
            const int e = l + k * TP;
            if (e < NA * NB) sm[(e / NA) * TL::RS + (e % NA)] = f[e];
        }
    }
    __syncthreads();
    if (on_x) {
        cx<T> v[LA::NL];
#pragma unroll
        for (int i = 0; i < LA::NL; i++) v[i] = sm[yb * TL::RS + LA::nat(i, hb)];
        LA::template dif<+1>(v, hb, mx);
#pragma unroll
        for (int q = 0; q < LA::NL; q++) sm[yb * TL::RS + LA::slot(q, hb)] = v[q];
    }
    __syncthreads();
    if (on_y) {
        cx<T> v[LB::NL];
#pragma unroll
        for (int i = 0; i < LB::NL; i++) v[i] = sm[LB::nat(i, ha) * TL::RS + xa];
        LB::template dif<+1>(v, ha, my);
#pragma unroll
        for (int q = 0; q < LB::NL; q++) sm[LB::slot(q, ha) * TL::RS + xa] = v[q];
    }
    __syncthreads();
    if (ok) {
        constexpr int EB = (ACC || LGF_EPI_ALL) ? LGF_EPI_BATCH : 1;
        for (int i0 = t; i0 < NA * NB; i0 += EB * TG) {
            cx<T> Gold[EB][6];
            if (ACC) {
#pragma unroll
                for (int b = 0; b < EB; b++)
                    if (i0 + b * TG < NA * NB) {
#pragma unroll
                        for (int k = 0; k < 6; k++) Gold[b][k] = gbuf[(int64_t)k * V + base + i0 + b * TG];
                    }
            }
#pragma unroll
            for (int b = 0; b < EB; b++) {
                const int i = i0 + b * TG;
                if (i < NA * NB) {
                    const int o = (i / NA) * TL::RS + (i % NA);
                    cx<T> g[9];
                    m_from_packed<T>(smp[o], smp[TL::ELEMS + o], smp[2 * TL::ELEMS + o], smp[3 * TL::ELEMS + o], a, g);
                    finish_g01<T>(g, gexp);
                    emit_g<T, ACC>(g, Gold[b], gbuf + base + i, V);
                }
            }
        }
    }
}

// The same pass for planes whose four fields do not fit one SM's shared memory (64^2 in FP64:
// 266 KB): a thread-block CLUSTER of LGF_XYG_CLUSTER CTAs holds the plane, 4 / LGF_XYG_CLUSTER fields each; after the
// transforms each CTA builds g for its share of the sites, reading its own fields locally and
// the others from the peers' shared memory (DSMEM).
// LGF_XYG_CLUSTER: CTAs per cluster, 2 (two fields per CTA, one CTA per SM for 64^2 FP64 planes) or 4 (one field per CTA,
// three CTAs per SM; each CTA then reads three of the four fields of its quarter of the sites through DSMEM).
// Same-run A/B in profiles/r02_xyg_cluster.md.
#ifndef LGF_XYG_CLUSTER
#define LGF_XYG_CLUSTER 4   /* 64^4 FP64: 792 us against 827 us with 2 (profiles/r02_xyg_cluster.md) */
#endif
template <typename T, int NA, int NB> struct XYG2Cfg {
    typedef Tile<NA, NB, 1, split_min<T>(NA, NB)> TL;
    static constexpr int CS = LGF_XYG_CLUSTER, FPC = 4 / CS;  // cluster size, fields per CTA
    static_assert(CS == 2 || CS == 4, "LGF_XYG_CLUSTER must be 2 or 4");
    static constexpr int TP = (TL::SA > 1 || TL::SB > 1) ? (TL::THREADS + 31) / 32 * 32 : TL::THREADS;
    static constexpr int CTA = FPC * TP;
    static constexpr size_t SMEM = (size_t)FPC * TL::ELEMS * sizeof(cx<T>);
    static constexpr bool FITS = SMEM <= 227 * 1024 && CTA <= 1024 && CTA >= 64;
};

template <typename T, int NA, int NB, bool ACC>
__global__ void __cluster_dims__(LGF_XYG_CLUSTER, 1, 1) __launch_bounds__((XYG2Cfg<T, NA, NB>::CTA))
k_fft_xy_inv_g2(const cx<T> *__restrict__ w, cx<T> *__restrict__ gbuf, int64_t V, T a, int gexp, const Ctrl *ctrl)
{
    namespace cg = cooperative_groups;
    if (*(volatile const int *)&ctrl->done) return;          // uniform over the grid: both CTAs of a cluster leave
    typedef XYG2Cfg<T, NA, NB> CF;
    typedef typename CF::TL TL;
    typedef Line<T, NA, TL::SA> LA;
    typedef Line<T, NB, TL::SB> LB;
    constexpr int TP = CF::TP;
    cg::cluster_group cluster = cg::this_cluster();
    constexpr int CS = CF::CS, FPC = CF::FPC;
    const int rank = (int)cluster.block_rank();              // fields [rank FPC, (rank + 1) FPC)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T> *smp = (cx<T> *)smem_raw;
    const int t = threadIdx.x, lf = t / TP, l = t % TP;
    cx<T> *sm = smp + (size_t)lf * TL::ELEMS;
    const int64_t plane = blockIdx.x / CS;
    const int64_t base = plane * (int64_t)(NA * NB);
    int xa, ha, yb, hb;
    line_of_thread<TL::SB>(l, xa, ha);
    line_of_thread<TL::SA>(l, yb, hb);
    const bool on_y = xa < NA && l < TL::SB * NA, on_x = yb < NB && l < TL::SA * NB;
    const unsigned my = __ballot_sync(0xffffffffu, on_y), mx = __ballot_sync(0xffffffffu, on_x);
    {
        const cx<T> *f = w + (int64_t)(FPC * rank + lf) * V + base;
#pragma unroll
        for (int k = 0; k < (NA * NB + TP - 1) / TP; k++) {
            const int e = l + k * TP;
            if (e < NA * NB) sm[(e / NA) * TL::RS + (e % NA)] = f[e];
        }
    }
    __syncthreads();
    if (on_x) {
        cx<T> v[LA::NL];
#pragma unroll
        for (int i = 0; i < LA::NL; i++) v[i] = sm[yb * TL::RS + LA::nat(i, hb)];
        LA::template dif<+1>(v, hb, mx);
#pragma unroll
        for (int q = 0; q < LA::NL; q++) sm[yb * TL::RS + LA::slot(q, hb)] = v[q];
    }
    __syncthreads();
    if (on_y) {
        cx<T> v[LB::NL];
#pragma unroll
        for (int i = 0; i < LB::NL; i++) v[i] = sm[LB::nat(i, ha) * TL::RS + xa];
        LB::template dif<+1>(v, ha, my);
#pragma unroll
        for (int q = 0; q < LB::NL; q++) sm[LB::slot(q, ha) * TL::RS + xa] = v[q];
    }
    cluster.sync();                                          // all four fields of the plane are in place
    // field k of the plane lives in CTA k / FPC at slot k % FPC (this CTA's own fields through its own mapping)
    const cx<T> *fld[4];
#pragma unroll
    for (int k = 0; k < 4; k++) fld[k] = cluster.map_shared_rank(smp, k / FPC) + (size_t)(k % FPC) * TL::ELEMS;
    constexpr int HALF = NA * NB / CS;                       // this CTA's share of the sites
    constexpr int EB = (ACC || LGF_EPI_ALL) ? LGF_EPI_BATCH : 1;
    for (int i0 = rank * HALF + t; i0 < (rank + 1) * HALF; i0 += EB * CF::CTA) {
        cx<T> Gold[EB][6];
        if (ACC) {
#pragma unroll
            for (int b = 0; b < EB; b++)
                if (i0 + b * CF::CTA < (rank + 1) * HALF) {
#pragma unroll
                    for (int k = 0; k < 6; k++) Gold[b][k] = gbuf[(int64_t)k * V + base + i0 + b * CF::CTA];
                }
        }
#pragma unroll
        for (int b = 0; b < EB; b++) {
            const int i = i0 + b * CF::CTA;
            if (i < (rank + 1) * HALF) {
                const int o = (i / NA) * TL::RS + (i % NA);
                cx<T> g[9];
                m_from_packed<T>(fld[0][o], fld[1][o], fld[2][o], fld[3][o], a, g);
                finish_g01<T>(g, gexp);
                emit_g<T, ACC>(g, Gold[b], gbuf + base + i, V);
            }
        }
    }
    cluster.sync();                                          // the peer may still be reading this CTA's fields
}

// ---------------------------------------------------------------- 1D passes along z or t
// One line per thread (or pair of lanes), consecutive threads on consecutive x: the 1D passes of the
// 4 x 1D structure (LGF_OPT_FFT_PASSES = 8).  Natural order in, natural order out, in place.  MASK: the
// t-forward pass also applies p_max^2/(p^2 V), zero mode -> 0 (eq. 1.2).
template <typename T, int N, int S, int SIGN, bool MASK>
__global__ void __launch_bounds__(256)
k_fft_axis(cx<T> *__restrict__ w, Geom geo, int axis, int64_t nlines, const double *__restrict__ ptab, double pmax2_over_V, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    typedef Line<T, N, S> LN;
    int ll, h;
    line_of_thread<S>((int)threadIdx.x, ll, h);
    const int64_t line = (int64_t)blockIdx.x * (256 / S) + ll;
    const bool on = line < nlines;
    const unsigned m = __ballot_sync(0xffffffffu, on);
    if (!on) return;
    // line -> (x, y, the other of z / t, field); axis = 2: lines along z, axis = 3: lines along t
    const int Nx = geo.N[0], Ny = geo.N[1], No = geo.N[axis == 2 ? 3 : 2];
    unsigned u = (unsigned)line;
    const int x = (int)(u % (unsigned)Nx); u /= (unsigned)Nx;
    const int y = (int)(u % (unsigned)Ny); u /= (unsigned)Ny;
    const int o = (int)(u % (unsigned)No); u /= (unsigned)No;
    const int64_t so = geo.st[axis == 2 ? 3 : 2], sa = geo.st[axis];
    cx<T> *f = w + (int64_t)u * geo.V + x + (int64_t)Nx * y + so * o;
    cx<T> v[LN::NL];
#pragma unroll
    for (int i = 0; i < LN::NL; i++) v[i] = f[sa * LN::nat(i, h)];
    LN::template dif<SIGN>(v, h, m);
    if (MASK) {
        const int z = axis == 2 ? 0 : o;                 // MASK runs on t-lines only (axis = 3): o is z
        const double pxyz = ptab[x] + ptab[Nx + y] + ptab[Nx + Ny + z];
        const double *pt = ptab + Nx + Ny + geo.N[2];
#pragma unroll
        for (int q = 0; q < LN::NL; q++) v[q] = cscale(v[q], (T)mask_factor(pmax2_over_V, pxyz + pt[LN::slot(q, h)]));
    }
#pragma unroll
    for (int q = 0; q < LN::NL; q++) f[sa * LN::slot(q, h)] = v[q];
}

template <typename T, int N> static int launch_axis_n(const FftArgs &a, int axis, int sign, int mask, cudaStream_t st)
{
    constexpr int S = split_of(N, split_min<T>(N, N));
    const int64_t nlines = (int64_t)a.nfields * a.geo.V / N;
    const unsigned grid = (unsigned)((nlines + 256 / S - 1) / (256 / S));
    const double c = a.pmax2 / a.vnorm;
    if (sign < 0 && mask) k_fft_axis<T, N, S, -1, true><<<grid, 256, 0, st>>>((cx<T> *)a.w, a.geo, axis, nlines, a.ptab, c, a.ctrl);
    else if (sign < 0) k_fft_axis<T, N, S, -1, false><<<grid, 256, 0, st>>>((cx<T> *)a.w, a.geo, axis, nlines, a.ptab, c, a.ctrl);
    else k_fft_axis<T, N, S, +1, false><<<grid, 256, 0, st>>>((cx<T> *)a.w, a.geo, axis, nlines, a.ptab, c, a.ctrl);
    return 0;
}

// ---------------------------------------------------------------- dispatch
template <typename T, int N> static int setup_xy_n()
{
    cudaError_t e;
    e = cudaFuncSetAttribute(k_fft_xy<T, N, N, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYCfg<T, N, N>::SMEM);
    if (e != cudaSuccess) return 1;
    e = cudaFuncSetAttribute(k_fft_xy<T, N, N, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYCfg<T, N, N>::SMEM);
    if (e != cudaSuccess) return 1;
    e = cudaFuncSetAttribute(k_fft_xy<T, N, N, 0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYCfg<T, N, N>::SMEM);
    if (e != cudaSuccess) return 1;
    e = cudaFuncSetAttribute(k_fft_xy<T, N, N, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYCfg<T, N, N>::SMEM);
    if (e != cudaSuccess) return 1;
    if (XYGCfg<T, N, N>::FITS) {
        e = cudaFuncSetAttribute(k_fft_xy_inv_g<T, N, N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYGCfg<T, N, N>::SMEM);
        if (e != cudaSuccess) return 1;
        e = cudaFuncSetAttribute(k_fft_xy_inv_g<T, N, N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYGCfg<T, N, N>::SMEM);
        if (e != cudaSuccess) return 1;
    } else if (XYG2Cfg<T, N, N>::FITS) {
        e = cudaFuncSetAttribute(k_fft_xy_inv_g2<T, N, N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYG2Cfg<T, N, N>::SMEM);
        if (e != cudaSuccess) return 1;
        e = cudaFuncSetAttribute(k_fft_xy_inv_g2<T, N, N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYG2Cfg<T, N, N>::SMEM);
        if (e != cudaSuccess) return 1;
    }
    return 0;
}

template <typename T, int N> static int launch_xy_n(const FftArgs &a, int which, cudaStream_t st)
{
    typedef XYCfg<T, N, N> X;
    const int64_t nplanes = (int64_t)a.nfields * a.geo.N[2] * a.geo.N[3];
    const unsigned grid = (unsigned)((nplanes + X::G - 1) / X::G);
    if (which == 0) k_fft_xy<T, N, N, 0><<<grid, X::CTA, X::SMEM, st>>>((cx<T> *)a.w, nplanes, a.ctrl);
    else k_fft_xy<T, N, N, 1><<<grid, X::CTA, X::SMEM, st>>>((cx<T> *)a.w, nplanes, a.ctrl);
    return 0;
}
// 1D passes along x (ax = 1) or y (ax = 2), forward (inverse = 0) or inverse
template <typename T, int N> static int launch_xy1d_n(const FftArgs &a, int inverse, int ax, cudaStream_t st)
{
    typedef XYCfg<T, N, N> X;
    const int64_t nplanes = (int64_t)a.nfields * a.geo.N[2] * a.geo.N[3];
    const unsigned grid = (unsigned)((nplanes + X::G - 1) / X::G);
    if (!inverse && ax == 1) k_fft_xy<T, N, N, 0, 1><<<grid, X::CTA, X::SMEM, st>>>((cx<T> *)a.w, nplanes, a.ctrl);
    else if (!inverse) k_fft_xy<T, N, N, 0, 2><<<grid, X::CTA, X::SMEM, st>>>((cx<T> *)a.w, nplanes, a.ctrl);
    else if (ax == 1) k_fft_xy<T, N, N, 1, 1><<<grid, X::CTA, X::SMEM, st>>>((cx<T> *)a.w, nplanes, a.ctrl);
    else k_fft_xy<T, N, N, 1, 2><<<grid, X::CTA, X::SMEM, st>>>((cx<T> *)a.w, nplanes, a.ctrl);
    return 0;
}

template <typename T, int N> static int launch_inv_g_n(const FftArgs &a, void *gbuf, double alpha, int gexp, int accum, cudaStream_t st)
{
    const int64_t nplanes = (int64_t)a.geo.N[2] * a.geo.N[3];
    if (XYGCfg<T, N, N>::FITS) {
        typedef XYGCfg<T, N, N> X;
        const unsigned grid = (unsigned)((nplanes + X::G - 1) / X::G);
        if (accum) k_fft_xy_inv_g<T, N, N, true><<<grid, X::CTA, X::SMEM, st>>>((const cx<T> *)a.w, (cx<T> *)gbuf, a.geo.V, nplanes, (T)(alpha / 2.0), gexp, a.ctrl);
        else k_fft_xy_inv_g<T, N, N, false><<<grid, X::CTA, X::SMEM, st>>>((const cx<T> *)a.w, (cx<T> *)gbuf, a.geo.V, nplanes, (T)(alpha / 2.0), gexp, a.ctrl);
    } else {
        typedef XYG2Cfg<T, N, N> X;                           // one cluster of two CTAs per plane
        if (accum) k_fft_xy_inv_g2<T, N, N, true><<<(unsigned)(X::CS * nplanes), X::CTA, X::SMEM, st>>>((const cx<T> *)a.w, (cx<T> *)gbuf, a.geo.V, (T)(alpha / 2.0), gexp, a.ctrl);
        else k_fft_xy_inv_g2<T, N, N, false><<<(unsigned)(X::CS * nplanes), X::CTA, X::SMEM, st>>>((const cx<T> *)a.w, (cx<T> *)gbuf, a.geo.V, (T)(alpha / 2.0), gexp, a.ctrl);
    }
    return 0;
}

template <typename T, int N> static int gbuf_fits_n() { return (XYGCfg<T, N, N>::FITS || XYG2Cfg<T, N, N>::FITS) ? 1 : 0; }

// Lattices with Nx = Ny and every extent in {8, 12, 16, 24, 32, 48, 64}: the (x,y) passes are instantiated
// per Nx (= Ny) and the (z,t) pass per (Nz, Nt) pair (fft_zt_inst.cu, one translation unit per Nz), which
// covers the cubic lattices, the N_s^3 x N_t shapes (16^3 x 32, 24^3 x 48, the paper's 32^3 x n)
// and (x,y) != (z,t) shapes alike.  The x-columns of a (z,t) tile (2, 4 or 8, chosen per (precision, Nz,
// Nt)) must divide Nx; the one family that fails this, FP32 with Nx = 12 and Nz != 12, takes the generic path
// like every other extent.
#define LGF_ZT_DECL(N)                                            \
    int zt_columns_na##N(int nt, int prec);                       \
    int zt_setup_na##N(int nt, int prec);                         \
    int zt_launch_na##N(const FftArgs &a, cudaStream_t st);       \
    int zt_has_half_na##N(int nt);                                \
    int zt_launch_half_na##N(const FftArgs &a, int inverse, cudaStream_t st);
LGF_ZT_DECL(8) LGF_ZT_DECL(12) LGF_ZT_DECL(16) LGF_ZT_DECL(24) LGF_ZT_DECL(32) LGF_ZT_DECL(48) LGF_ZT_DECL(64)
#undef LGF_ZT_DECL
#define LGF_NZ_SWITCH(FN, ...)                \
    switch (nz) {                             \
    case 8: return FN##8(__VA_ARGS__);        \
    case 12: return FN##12(__VA_ARGS__);      \
    case 16: return FN##16(__VA_ARGS__);      \
    case 24: return FN##24(__VA_ARGS__);      \
    case 32: return FN##32(__VA_ARGS__);      \
    case 48: return FN##48(__VA_ARGS__);      \
    case 64: return FN##64(__VA_ARGS__);      \
    default: break;                           \
    }
static int zt_columns(int nz, int nt, int prec)
{
    LGF_NZ_SWITCH(zt_columns_na, nt, prec)
    return 0;
}
static bool tiled_extent(int n) { return n == 8 || n == 16 || n == 32 || n == 64 || n == 12 || n == 24 || n == 48; }
bool fft_tiled_supported(const int N[4], int prec)
{
    if (!(N[0] == N[1] && tiled_extent(N[0]) && tiled_extent(N[2]) && tiled_extent(N[3]))) return false;
    const int c = zt_columns(N[2], N[3], prec);
    return c > 0 && N[0] % c == 0;
}
int fft_tiled_zt_columns(const int N[4], int prec) { return fft_tiled_supported(N, prec) ? zt_columns(N[2], N[3], prec) : 0; }

#define LGF_FFT_SWITCH(FN, ...)                                         \
    switch (n) {                                                        \
    case 8: return prec == 0 ? FN<double, 8>(__VA_ARGS__) : FN<float, 8>(__VA_ARGS__);    \
    case 12: return prec == 0 ? FN<double, 12>(__VA_ARGS__) : FN<float, 12>(__VA_ARGS__); \
    case 16: return prec == 0 ? FN<double, 16>(__VA_ARGS__) : FN<float, 16>(__VA_ARGS__); \
    case 24: return prec == 0 ? FN<double, 24>(__VA_ARGS__) : FN<float, 24>(__VA_ARGS__); \
    case 32: return prec == 0 ? FN<double, 32>(__VA_ARGS__) : FN<float, 32>(__VA_ARGS__); \
    case 48: return prec == 0 ? FN<double, 48>(__VA_ARGS__) : FN<float, 48>(__VA_ARGS__); \
    case 64: return prec == 0 ? FN<double, 64>(__VA_ARGS__) : FN<float, 64>(__VA_ARGS__); \
    default: break;                                                     \
    }

static int setup_xy(int n, int prec)
{
    LGF_FFT_SWITCH(setup_xy_n)
    return 1;
}
static int setup_zt(int nz, int nt, int prec)
{
    LGF_NZ_SWITCH(zt_setup_na, nt, prec)
    return 1;
}
int fft_tiled_setup(const int N[4], int prec) { return setup_xy(N[0], prec) | setup_zt(N[2], N[3], prec); }

// does the plane of 4 packed fields fit in shared memory (pass 2 with the g build fused)?
bool fft_tiled_gbuf_supported(const int N[4], int prec)
{
    if (!fft_tiled_supported(N, prec)) return false;
    const int n = N[0];
    LGF_FFT_SWITCH(gbuf_fits_n)
    return false;
}

static int run_xy(const FftArgs &a, int which, cudaStream_t st)
{
    const int n = a.geo.N[0], prec = a.prec;
    LGF_FFT_SWITCH(launch_xy_n, a, which, st)
    return 1;
}
static int run_zt(const FftArgs &a, cudaStream_t st)
{
    const int nz = a.geo.N[2];
    LGF_NZ_SWITCH(zt_launch_na, a, st)
    return 1;
}
void launch_fft_tiled(const FftArgs &a, int which, cudaStream_t st)
{
    if (which == 1) run_zt(a, st); else run_xy(a, which, st);
}

// ---- the other pass structures of the paper's comparison (LGF_OPT_FFT_PASSES)
static int run_xy1d(const FftArgs &a, int inverse, int ax, cudaStream_t st)
{
    const int n = a.geo.N[0], prec = a.prec;
    LGF_FFT_SWITCH(launch_xy1d_n, a, inverse, ax, st)
    return 1;
}
static int run_axis(const FftArgs &a, int axis, int sign, int mask, cudaStream_t st)
{
    const int n = a.geo.N[axis], prec = a.prec;
    LGF_FFT_SWITCH(launch_axis_n, a, axis, sign, mask, st)
    return 1;
}
static int run_zt_half(const FftArgs &a, int inverse, cudaStream_t st)
{
    const int nz = a.geo.N[2];
    LGF_NZ_SWITCH(zt_launch_half_na, a, inverse, st)
    return 1;
}
bool fft_tiled_passes_supported(const int N[4], int prec, int passes)
{
    if (!fft_tiled_supported(N, prec)) return false;
    if (passes == 3 || passes == 8) return true;
    if (passes == 4) { const int nz = N[2]; LGF_NZ_SWITCH(zt_has_half_na, N[3]) return false; }
    return false;
}
// 2D + 2D as four passes (the paper's best): step 0 (x,y) forward, 1 (z,t) forward times the mask,
// 2 (z,t) inverse, 3 (x,y) inverse (or launch_fft_tiled_inv_g in its place)
void launch_fft_tiled_4pass(const FftArgs &a, int step, cudaStream_t st)
{
    if (step == 0) run_xy(a, 0, st);
    else if (step == 1) run_zt_half(a, 0, st);
    else if (step == 2) run_zt_half(a, 1, st);
    else run_xy(a, 2, st);
}
// 4 x 1D as eight passes: steps 0..3 forward along y, x, z, t (the mask rides on the last), 4..7 inverse along t, z, x, y
void launch_fft_tiled_8pass(const FftArgs &a, int step, cudaStream_t st)
{
    switch (step) {
    case 0: run_xy1d(a, 0, 2, st); break;
    case 1: run_xy1d(a, 0, 1, st); break;
    case 2: run_axis(a, 2, -1, 0, st); break;
    case 3: run_axis(a, 3, -1, 1, st); break;
    case 4: run_axis(a, 3, +1, 0, st); break;
    case 5: run_axis(a, 2, +1, 0, st); break;
    case 6: run_xy1d(a, 1, 1, st); break;
    default: run_xy1d(a, 1, 2, st); break;
    }
}

// pass 2 fused with the g build: needs the 4 packed fields (nfields == 4)
static int run_inv_g(const FftArgs &a, void *gbuf, double alpha, int gexp, int accum, cudaStream_t st)
{
    const int n = a.geo.N[0], prec = a.prec;
    LGF_FFT_SWITCH(launch_inv_g_n, a, gbuf, alpha, gexp, accum, st)
    return 1;
}
void launch_fft_tiled_inv_g(const FftArgs &a, void *gbuf, double alpha, int gexp, int accum, cudaStream_t st) { run_inv_g(a, gbuf, alpha, gexp, accum, st); }

} // namespace lgf
