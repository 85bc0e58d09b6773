// fft_zt.cuh -- pass 1 of the tiled FFT (Alg. 1 lines 3-8): (z,t) forward, times
// p_max^2/(p^2 V) (eq. 1.2; zero mode -> 0), (z,t) inverse, one visit per tile.
// Kernel templates and their launchers; instantiated per Nz by fft_zt_inst.cu (one translation unit
// per Nz so that the 7 x 7 (Nz, Nt) pairs compile in parallel), dispatched from fft_tiled.cu.
#pragma once
#include "fft_lines.cuh"

namespace lgf {

// ---------------------------------------------------------------- pass 1: (z,t) tiles
// Tile = C consecutive x at fixed (field, y): element (c, z, t) at global x0 + c + sz*z + st*t.
// z-lines straight from global (thread = (c, t)), Dif(-) along z -> shared; t-lines from
// shared (thread = (c, kz)): Dif(-), mask, Dit(+) -> shared; z-lines from shared: Dif(+),
// stored straight to global.  p^2 = sum_mu 4 sin^2(pi k_mu/N_mu) (reading R5) from the
// per-axis tables; the factor p_max^2/(p^2 V) is one FP64 division per mode.
// Timing-only experiment on k_fft_zt (WRONG results; profiles/r02_zt_phases.md): 1 = memory only (every global and shared
// load / store of the pass, no transform, no mask), 2 = arithmetic only (no global loads or stores; shared memory kept).
#ifndef LGF_ZT_EXP
#define LGF_ZT_EXP 0
#endif
#ifndef LGF_ZT_MAXB
#define LGF_ZT_MAXB 2   /* 3 measured slower at 32^4 (47.6 vs 45.5 us: spills), equal at 48^4 */
#endif
// 16- or 8-byte asynchronous copy global -> shared (LDGSTS): the data is in flight without holding registers
template <typename V> __device__ __forceinline__ void cp_async_elem(V *smem_dst, const V *gsrc)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    if (sizeof(V) == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gsrc) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
template <typename T, int NA, int NB, int C> struct ZTCfg {
    typedef Tile<NA, NB, C, split_min<T>(NA, NB)> TL;
    static constexpr int TT = TL::THREADS;
    static constexpr int CTA = cta_threads(TT);
    static constexpr int G = CTA / TT;
    static constexpr size_t PT = ((NB * sizeof(double) + 15) / 16) * 16;
    static constexpr size_t SMEM = PT + (size_t)G * TL::ELEMS * sizeof(cx<T>);
    // CTAs per SM that shared memory allows (1 KB reserved each); registers are capped to match
    static constexpr int FIT = (int)((size_t)227 * 1024 / (SMEM + 1024));
    static constexpr int MINB0 = FIT < 1 ? 1 : (FIT > LGF_ZT_MAXB ? LGF_ZT_MAXB : FIT);
    // 32-bit registers that the longest line of a thread needs for its data alone; when that already reaches the
    // register cap of MINB0 CTAs per SM (mixed tiles such as 16 x 64: 32 FP64 complex numbers per thread against
    // 128 registers) the transforms would run out of local memory, so such tiles run one CTA per SM
    static constexpr int NLA = NA / TL::SA, NLB = NB / TL::SB;
    static constexpr int DATA = (NLA > NLB ? NLA : NLB) * (int)(sizeof(cx<T>) / 4);
    static constexpr int MINB = (MINB0 > 1 && DATA >= 65536 / (CTA * MINB0)) ? 1 : MINB0;
};

template <typename T, int NA, int NB, int C>
__global__ void __launch_bounds__((ZTCfg<T, NA, NB, C>::CTA), (ZTCfg<T, NA, NB, C>::MINB))
k_fft_zt(cx<T> *__restrict__ w, Geom geo, const double *__restrict__ ptab, double pmax2_over_V, int64_t ntiles, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    typedef ZTCfg<T, NA, NB, C> CF;
    typedef typename CF::TL TL;
    typedef Line<T, NA, TL::SA> LA;
    typedef Line<T, NB, TL::SB> LB;
    constexpr int TT = CF::TT, G = CF::G;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *pt = (double *)smem_raw;                                  // 4 sin^2(pi kt/Nt), NB entries
    cx<T> *sm0 = (cx<T> *)(smem_raw + CF::PT);
    const int grp = threadIdx.x / TT, t = threadIdx.x % TT;
    cx<T> *sm = sm0 + (size_t)grp * TL::ELEMS;
    const int64_t tile = (int64_t)blockIdx.x * G + grp;
    const bool ok = tile < ntiles && grp < G;
    const int Nx = geo.N[0], Ny = geo.N[1];
    const int xchunks = Nx / C;
    // tile -> (field, y, xchunk)
    const int xc = (int)(tile % xchunks);
    const int y = (int)((tile / xchunks) % Ny);
    const int64_t fld = tile / ((int64_t)xchunks * Ny);
    const int x0 = xc * C;
    cx<T> *f = w + fld * geo.V + x0 + (int64_t)Nx * y;
    const int64_t sz = geo.st[2], st = geo.st[3];
    for (int i = threadIdx.x; i < NB; i += CF::CTA) pt[i] = ptab[Nx + Ny + NA + i];
    int la, ha, lb, hb;                                                // z-line (c, t) / t-line (c, kz) of this thread
    line_of_thread<TL::SA>(t, la, ha);
    line_of_thread<TL::SB>(t, lb, hb);
    const int ca = la % C, ta = la / C, cb = lb % C, zb = lb / C;
    const bool on_z = ok && ta < NB && t < TL::SA * C * NB, on_t = ok && zb < NA && t < TL::SB * C * NA;
    const unsigned mz = __ballot_sync(0xffffffffu, on_z), mt = __ballot_sync(0xffffffffu, on_t);

    if (on_z) {                                                        // z-line at (c, t) = (ca, ta)
        cx<T> v[LA::NL];
        const cx<T> *g = f + ca + st * ta;
#pragma unroll
        for (int i = 0; i < LA::NL; i++) v[i] = LGF_ZT_EXP == 2 ? mk<T>((T)(t + i) * (T)1e-3, (T)(i - t) * (T)1e-3) : g[sz * LA::nat(i, ha)];
        if (LGF_ZT_EXP != 1) LA::template dif<-1>(v, ha, mz);
#pragma unroll
        for (int q = 0; q < LA::NL; q++) sm[ta * TL::RS + LA::slot(q, ha) * C + ca] = v[q];
    }
    __syncthreads();
    if (on_t) {                                                        // t-line at (c, kz) = (cb, zb)
        cx<T> v[LB::NL];
#pragma unroll
        for (int i = 0; i < LB::NL; i++) v[i] = sm[LB::nat(i, hb) * TL::RS + zb * C + cb];
        if (LGF_ZT_EXP != 1) LB::template dif<-1>(v, hb, mt);
        const double pxyz = ptab[x0 + cb] + ptab[Nx + y] + ptab[Nx + Ny + zb];
        if (LGF_ZT_EXP != 1) {
#pragma unroll
        for (int q = 0; q < LB::NL; q++) {
            const T fac = (T)mask_factor(pmax2_over_V, pxyz + pt[LB::slot(q, hb)]);
            v[q] = cscale(v[q], fac);
        }
        LB::template dit<+1>(v, hb, mt);
        }
#pragma unroll
        for (int i = 0; i < LB::NL; i++) sm[LB::nat(i, hb) * TL::RS + zb * C + cb] = v[i];
    }
    __syncthreads();
    if (on_z) {
        cx<T> v[LA::NL];
#pragma unroll
        for (int i = 0; i < LA::NL; i++) v[i] = sm[ta * TL::RS + LA::nat(i, ha) * C + ca];
        if (LGF_ZT_EXP != 1) LA::template dif<+1>(v, ha, mz);
        cx<T> *g = f + ca + st * ta;
#pragma unroll
        for (int q = 0; q < LA::NL; q++) if (LGF_ZT_EXP != 2 || v[q].x == (T)123456.789) g[sz * LA::slot(q, ha)] = v[q];
    }
}

// The same pass as a PERSISTENT kernel with register-free prefetch (LGF_OPT_ZT_PIPE): a thread group walks
// the tiles  first, first + stride, ...  and keeps its shared-memory tile for all of them.  The z-line a
// thread transforms first (forward) and last (inverse) is the same line of every tile, so right after
// it has read its inverse-transform input out of shared memory it issues the asynchronous copies
// (cp.async, 16 bytes each) of the SAME elements of the next tile into the SAME shared-memory slots:
// they land while this thread finishes the inverse transform and its stores, and while the rest of
// the CTA is still at work, and no register is held for data in flight.  At the top of the next tile
// each thread waits for its own copies only (cp.async.wait_all): no barrier is needed for the hand-over
// because the slots are private to the thread (pair of lanes for split lines) between the two
// barriers of a tile.  In k_fft_zt every tile starts with a cold load -> transform -> store
// sequence and only the other CTA on the SM hides it (ncu, profiles/r01e_final.md: 23 % warps active).
template <typename T, int NA, int NB, int C>
__global__ void __launch_bounds__((ZTCfg<T, NA, NB, C>::CTA), (ZTCfg<T, NA, NB, C>::MINB))
k_fft_zt_pipe(cx<T> *__restrict__ w, Geom geo, const double *__restrict__ ptab, double pmax2_over_V, int64_t ntiles, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    typedef ZTCfg<T, NA, NB, C> CF;
    typedef typename CF::TL TL;
    typedef Line<T, NA, TL::SA> LA;
    typedef Line<T, NB, TL::SB> LB;
    constexpr int TT = CF::TT, G = CF::G;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *pt = (double *)smem_raw;
    cx<T> *sm0 = (cx<T> *)(smem_raw + CF::PT);
    const int grp = threadIdx.x / TT, t = threadIdx.x % TT;
    cx<T> *sm = sm0 + (size_t)grp * TL::ELEMS;
    const int Nx = geo.N[0], Ny = geo.N[1];
    const int xchunks = Nx / C;
    const int64_t sz = geo.st[2], st = geo.st[3];
    for (int i = threadIdx.x; i < NB; i += CF::CTA) pt[i] = ptab[Nx + Ny + NA + i];
    int la, ha, lb, hb;
    line_of_thread<TL::SA>(t, la, ha);
    line_of_thread<TL::SB>(t, lb, hb);
    const int ca = la % C, ta = la / C, cb = lb % C, zb = lb / C;
    const bool has_z = grp < G && ta < NB && t < TL::SA * C * NB, has_t = grp < G && zb < NA && t < TL::SB * C * NA;
    cx<T> *zrow = sm + ta * TL::RS + ca;                                // this thread's z-line in shared memory
    const int64_t stride = (int64_t)gridDim.x * G;
    // tile -> (field, y, xchunk) -> first element of the thread's z-line
    auto zline = [&](int64_t tile) -> cx<T> * {
        const int xc = (int)(tile % xchunks);
        const int y = (int)((tile / xchunks) % Ny);
        const int64_t fld = tile / ((int64_t)xchunks * Ny);
        return w + fld * geo.V + xc * C + (int64_t)Nx * y + ca + st * ta;
    };
    {
        const int64_t first = (int64_t)blockIdx.x * G + grp;
        if (has_z && first < ntiles) {
            const cx<T> *g = zline(first);
#pragma unroll
            for (int i = 0; i < LA::NL; i++) cp_async_elem(zrow + LA::nat(i, ha) * C, g + sz * LA::nat(i, ha));
        }
    }
    for (int64_t t0 = (int64_t)blockIdx.x * G; t0 < ntiles; t0 += stride) {
        const int64_t tile = t0 + grp;
        const bool ok = tile < ntiles;
        const bool on_z = ok && has_z, on_t = ok && has_t;
        const unsigned mz = __ballot_sync(0xffffffffu, on_z), mt = __ballot_sync(0xffffffffu, on_t);
        const int xc = (int)(tile % xchunks);
        const int y = (int)((tile / xchunks) % Ny);
        cp_async_wait_all();                                               // this thread's elements of the tile are in place
        if (on_z) {
            cx<T> v[LA::NL];
#pragma unroll
            for (int i = 0; i < LA::NL; i++) v[i] = zrow[LA::nat(i, ha) * C];
            LA::template dif<-1>(v, ha, mz);
#pragma unroll
            for (int q = 0; q < LA::NL; q++) zrow[LA::slot(q, ha) * C] = v[q];
        }
        __syncthreads();
        if (on_t) {
            cx<T> v[LB::NL];
#pragma unroll
            for (int i = 0; i < LB::NL; i++) v[i] = sm[LB::nat(i, hb) * TL::RS + zb * C + cb];
            LB::template dif<-1>(v, hb, mt);
            const double pxyz = ptab[xc * C + cb] + ptab[Nx + y] + ptab[Nx + Ny + zb];
#pragma unroll
            for (int q = 0; q < LB::NL; q++) {
                const T fac = (T)mask_factor(pmax2_over_V, pxyz + pt[LB::slot(q, hb)]);
                v[q] = cscale(v[q], fac);
            }
            LB::template dit<+1>(v, hb, mt);
#pragma unroll
            for (int i = 0; i < LB::NL; i++) sm[LB::nat(i, hb) * TL::RS + zb * C + cb] = v[i];
        }
        __syncthreads();
        if (on_z) {
            cx<T> v[LA::NL];
#pragma unroll
            for (int i = 0; i < LA::NL; i++) v[i] = zrow[LA::nat(i, ha) * C];
            if (tile + stride < ntiles) {                                  // next tile of this group: same slots
                const cx<T> *g = zline(tile + stride);
#pragma unroll
                for (int i = 0; i < LA::NL; i++) cp_async_elem(zrow + LA::nat(i, ha) * C, g + sz * LA::nat(i, ha));
            }
            LA::template dif<+1>(v, ha, mz);
            cx<T> *g = zline(tile);
#pragma unroll
            for (int q = 0; q < LA::NL; q++) g[sz * LA::slot(q, ha)] = v[q];
        }
    }
    cp_async_wait_all();
}

// ---------------------------------------------------------------- the (z,t) pass as two launches
// 2D + 2D without the fusion of the middle (the structure the paper found best with CUFFT, PAPER.md:119:
// "two 2D FFTs"; LGF_OPT_FFT_PASSES = 4): INVERSE = 0 transforms a tile forward along z and t and applies the
// mask, INVERSE = 1 transforms it back; the field crosses HBM once more than in k_fft_zt.  z-lines
// straight from global memory, through shared memory, t-lines stored straight to global memory;
// natural order in global memory on both sides.
template <typename T, int NA, int NB, int C, int INVERSE>
__global__ void __launch_bounds__((ZTCfg<T, NA, NB, C>::CTA), (ZTCfg<T, NA, NB, C>::MINB))
k_fft_zt_half(cx<T> *__restrict__ w, Geom geo, const double *__restrict__ ptab, double pmax2_over_V, int64_t ntiles, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    typedef ZTCfg<T, NA, NB, C> CF;
    typedef typename CF::TL TL;
    typedef Line<T, NA, TL::SA> LA;
    typedef Line<T, NB, TL::SB> LB;
    constexpr int TT = CF::TT, G = CF::G;
    constexpr int SIGN = INVERSE ? +1 : -1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *pt = (double *)smem_raw;
    cx<T> *sm0 = (cx<T> *)(smem_raw + CF::PT);
    const int grp = threadIdx.x / TT, t = threadIdx.x % TT;
    cx<T> *sm = sm0 + (size_t)grp * TL::ELEMS;
    const int64_t tile = (int64_t)blockIdx.x * G + grp;
    const bool ok = tile < ntiles && grp < G;
    const int Nx = geo.N[0], Ny = geo.N[1];
    const int xchunks = Nx / C;
    const int xc = (int)(tile % xchunks);
    const int y = (int)((tile / xchunks) % Ny);
    const int64_t fld = tile / ((int64_t)xchunks * Ny);
    const int x0 = xc * C;
    cx<T> *f = w + fld * geo.V + x0 + (int64_t)Nx * y;
    const int64_t sz = geo.st[2], st = geo.st[3];
    if (!INVERSE)
        for (int i = threadIdx.x; i < NB; i += CF::CTA) pt[i] = ptab[Nx + Ny + NA + i];
    int la, ha, lb, hb;
    line_of_thread<TL::SA>(t, la, ha);
    line_of_thread<TL::SB>(t, lb, hb);
    const int ca = la % C, ta = la / C, cb = lb % C, zb = lb / C;
    const bool on_z = ok && ta < NB && t < TL::SA * C * NB, on_t = ok && zb < NA && t < TL::SB * C * NA;
    const unsigned mz = __ballot_sync(0xffffffffu, on_z), mt = __ballot_sync(0xffffffffu, on_t);
    if (on_z) {
        cx<T> v[LA::NL];
        const cx<T> *g = f + ca + st * ta;
#pragma unroll
        for (int i = 0; i < LA::NL; i++) v[i] = g[sz * LA::nat(i, ha)];
        LA::template dif<SIGN>(v, ha, mz);
#pragma unroll
        for (int q = 0; q < LA::NL; q++) sm[ta * TL::RS + LA::slot(q, ha) * C + ca] = v[q];
    }
    __syncthreads();
    if (on_t) {
        cx<T> v[LB::NL];
#pragma unroll
        for (int i = 0; i < LB::NL; i++) v[i] = sm[LB::nat(i, hb) * TL::RS + zb * C + cb];
        LB::template dif<SIGN>(v, hb, mt);
        if (!INVERSE) {
            const double pxyz = ptab[x0 + cb] + ptab[Nx + y] + ptab[Nx + Ny + zb];
#pragma unroll
            for (int q = 0; q < LB::NL; q++) v[q] = cscale(v[q], (T)mask_factor(pmax2_over_V, pxyz + pt[LB::slot(q, hb)]));
        }
        cx<T> *g = f + cb + sz * zb;
#pragma unroll
        for (int q = 0; q < LB::NL; q++) g[st * LB::slot(q, hb)] = v[q];
    }
}

// ---------------------------------------------------------------- launchers
// x-columns per (z,t) tile: 64-byte runs in global memory (FP64), halved while the tile does not fit
// in shared memory or does not divide Nz.  The columns must also divide Nx, which the caller checks
// (zt_columns / fft_tiled_supported): a lattice whose Nx is not a multiple takes the generic transform.
#ifndef LGF_ZT_BYTES
#define LGF_ZT_BYTES 64
#endif
template <typename T, int NA, int NB> struct ZTC {
    static constexpr int WANT = LGF_ZT_BYTES / (int)sizeof(cx<T>);
    static constexpr size_t tile_bytes(int c) { return (size_t)(NA * c + c) * NB * sizeof(cx<T>); }
    static constexpr int C = tile_bytes(WANT) <= 200 * 1024 && NA % WANT == 0 ? WANT : (tile_bytes(WANT / 2) <= 200 * 1024 && NA % (WANT / 2) == 0 ? WANT / 2 : WANT / 4);
    static_assert(C >= 1 && tile_bytes(C) <= 220 * 1024, "(z,t) tile does not fit in shared memory");
};
// The persistent variant (LGF_OPT_ZT_PIPE) and the two-launch form (LGF_OPT_FFT_PASSES = 4) are instantiated
// for the square tiles and the 32 x n tiles of the paper's lattices only (measured slower than the plain kernel on every lattice tried, profiles/r02*);
// other pairs run the plain kernel whatever the option says.
constexpr bool zt_pipe_pair(int na, int nb) { return na == nb || (na == 32 && (nb == 8 || nb == 16 || nb == 48 || nb == 64)); }

template <typename T, int NA, int NB> int setup_zt_half_n();
template <typename T, int NA, int NB> int setup_zt_n()
{
    constexpr int C = ZTC<T, NA, NB>::C;
    typedef ZTCfg<T, NA, NB, C> Z;
    cudaError_t e = cudaFuncSetAttribute(k_fft_zt<T, NA, NB, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Z::SMEM);
    if (e != cudaSuccess) return 1;
    if constexpr (zt_pipe_pair(NA, NB)) {
        e = cudaFuncSetAttribute(k_fft_zt_pipe<T, NA, NB, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Z::SMEM);
        if (e != cudaSuccess) return 1;
    }
    return setup_zt_half_n<T, NA, NB>();
}

template <typename T, int NA, int NB> int setup_zt_half_n()
{
    if constexpr (zt_pipe_pair(NA, NB)) {
        constexpr int C = ZTC<T, NA, NB>::C;
        typedef ZTCfg<T, NA, NB, C> Z;
        if (cudaFuncSetAttribute(k_fft_zt_half<T, NA, NB, C, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Z::SMEM) != cudaSuccess) return 1;
        if (cudaFuncSetAttribute(k_fft_zt_half<T, NA, NB, C, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Z::SMEM) != cudaSuccess) return 1;
    }
    return 0;
}
template <typename T, int NA, int NB> int launch_zt_half_n(const FftArgs &a, int inverse, cudaStream_t st)
{
    if constexpr (zt_pipe_pair(NA, NB)) {
        constexpr int C = ZTC<T, NA, NB>::C;
        typedef ZTCfg<T, NA, NB, C> Z;
        const int64_t ntiles = (int64_t)a.nfields * a.geo.N[1] * (a.geo.N[0] / C);
        const unsigned grid = (unsigned)((ntiles + Z::G - 1) / Z::G);
        if (inverse) k_fft_zt_half<T, NA, NB, C, 1><<<grid, Z::CTA, Z::SMEM, st>>>((cx<T> *)a.w, a.geo, a.ptab, a.pmax2 / a.vnorm, ntiles, a.ctrl);
        else k_fft_zt_half<T, NA, NB, C, 0><<<grid, Z::CTA, Z::SMEM, st>>>((cx<T> *)a.w, a.geo, a.ptab, a.pmax2 / a.vnorm, ntiles, a.ctrl);
        return 0;
    }
    return 1;
}

inline int sm_count()
{
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
            cudaGetLastError();
            n = 148;
        }
    }
    return n;
}

template <typename T, int NA, int NB> int launch_zt_n(const FftArgs &a, cudaStream_t st)
{
    constexpr int C = ZTC<T, NA, NB>::C;
    typedef ZTCfg<T, NA, NB, C> Z;
    const int64_t ntiles = (int64_t)a.nfields * a.geo.N[1] * (a.geo.N[0] / C);
    const unsigned grid = (unsigned)((ntiles + Z::G - 1) / Z::G);
    if constexpr (zt_pipe_pair(NA, NB)) if (a.zt_pipe) {
        // persistent: as many CTAs as are resident at once, each walks tiles blockIdx, blockIdx + grid, ...
        const unsigned resident = (unsigned)(sm_count() * Z::MINB);
        k_fft_zt_pipe<T, NA, NB, C><<<grid < resident ? grid : resident, Z::CTA, Z::SMEM, st>>>((cx<T> *)a.w, a.geo, a.ptab, a.pmax2 / a.vnorm, ntiles, a.ctrl);
        return 0;
    }
    k_fft_zt<T, NA, NB, C><<<grid, Z::CTA, Z::SMEM, st>>>((cx<T> *)a.w, a.geo, a.ptab, a.pmax2 / a.vnorm, ntiles, a.ctrl);
    return 0;
}


} // namespace lgf
