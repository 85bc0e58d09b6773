// kernels_fused.cu -- kernel (c) and kernel (a) of the NEXT iteration in one pass over the links
// (arXiv 1210.8018, Alg. 1 lines 12-17):
//     U'_mu(x) = g(x) U_mu(x) g^dagger(x+mu)                       (stored, each link read once, written once)
//     Delta'(x) from  A'(x) = sum_nu [U'_nu(x-nu) - U'_nu(x)]      (eq. 1.5)
//     F', theta'                                                   (eq. 1.1, 1.4)
// The paper runs these as two kernels (k6, then k2 of the next iteration: Table 1,
// PAPER.md:146-150), so every link crosses the memory bus three times per iteration; here it
// crosses twice.  The thread of site x also needs the four NEW backward links
// U'_nu(x-nu) = g(x-nu) U_nu(x-nu) g^dagger(x); it recomputes what it needs of them from the OLD
// links (served by L2, they were or will be streamed by the thread of x-nu) instead of waiting
// for a grid-wide barrier.  That is why the links are double-buffered: `lin` is read-only,
// `lout` write-only.
// g comes from the g buffer written by the last FFT pass (GBUF) or is rebuilt from w.
#include "launch.h"
#include "su3.cuh"
#include "reduce.cuh"
#include <cstdio>
#include <cstdlib>
// 1: F and theta of the link kernel are summed in two levels (reduce.cuh, finish_measure_2l); 0: by the last block alone
#ifndef LGF_REDUCE_2L
#define LGF_REDUCE_2L 1
#endif
#ifndef LGF_FUSED_DUMMY_SMEM
#define LGF_FUSED_DUMMY_SMEM 0   /* experiment: dynamic shared memory the site kernel does not use (what a smaller L1 costs) */
#endif

namespace lgf {

#ifndef LGF_FUSED_THREADS
#define LGF_FUSED_THREADS 128
#endif
static const int FUSED_THREADS = LGF_FUSED_THREADS;
#ifndef LGF_FUSED_MINB
#define LGF_FUSED_MINB 4
#endif
// 1: the backward links are taken in the order t, z, y, x, so that the loads of U_x(x-x), g(x-x), g(x) and of
// the forward x-link that follows touch the same cache lines back to back (L1 hits instead of L2 hits).
// Same-run A/B on B200 (profiles/r02_link_kernel.md): 32^4 FP64 208.7 -> 203.1 us, 64^4 FP64 4488 -> 4358 us,
// 48^4 FP32 718 -> 723 us: on for FP64, off for FP32.
#ifndef LGF_FUSED_BWD_REV
#define LGF_FUSED_BWD_REV (sizeof(T) == 8)
#endif

// links are streamed: read (twice, the second time from L2) and written once per iteration
// tuning macros for the cache behaviour of the loads (same-run A/B, profiles/r02_link_kernel.md):
// LGF_LINK_LD: 0 ld.global.nc (default), 1 ld.global.nc.L1::no_allocate (the links are streamed; leave L1 to g)
#ifndef LGF_LINK_LD
#define LGF_LINK_LD 0
#endif
#ifndef LGF_FUSED_PREFETCH
#define LGF_FUSED_PREFETCH 0
#endif
__device__ __forceinline__ double2 ld_na(const double2 *p)
{
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 ld_na(const float2 *p)
{
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
template <typename V> __device__ __forceinline__ V ld_link(const V *p)
{
#if LGF_LINK_LD == 1
    return ld_na(p);
#else
    return __ldg(p);
#endif
}
// Link stores as st.global.cs (evict first): the new links are not read again before the next iteration, and
// written lines that linger in L2 push out the neighbour links and g that the kernel re-reads.  Same-run A/B on
// B200 (profiles/r02_link_kernel.md): FP64 32^4 12-real 211.2 -> 198.7 us, 32^4 18-real 273.2 -> 270.6, 64^4 4320 -> 4300,
// 16^4 23.6 -> 23.2; FP32 48^4 18-real 682.7 -> 708.6 (worse), 32^4 12-real 129.4 -> 127.8: on for FP64, off for FP32.
#ifndef LGF_LINK_STCS
#define LGF_LINK_STCS(V) (sizeof(V) == 16)
#endif
#ifndef LGF_W_EVICT_LAST
#define LGF_W_EVICT_LAST 0
#endif
template <typename V> __device__ __forceinline__ void st_link(V *p, V v)
{
    if (LGF_LINK_STCS(V)) __stcs(p, v); else *p = v;
}
// Delta is read back by the first FFT pass right after this kernel: ask L2 to keep it
__device__ __forceinline__ void st_field(double2 *p, double2 v)
{
#if LGF_W_EVICT_LAST
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
#else
    *p = v;
#endif
}
__device__ __forceinline__ void st_field(float2 *p, float2 v)
{
#if LGF_W_EVICT_LAST
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v.x), "f"(v.y), "l"(pol) : "memory");
#else
    *p = v;
#endif
}

template <typename T, int NE>
__device__ __forceinline__ void load_link_in(const cx<T> *__restrict__ links, int64_t V, int mu, int64_t s, cx<T> (&u)[9])
{
    const cx<T> *p = links + (int64_t)mu * NE * V + s;
#pragma unroll
    for (int k = 0; k < NE; k++) u[k] = ld_link(p + (int64_t)k * V);
    if (NE == 6) su3_row2(u);
}

// anti-Hermitian part of a link, accumulated with sign sg:  di += sg Im M_ii,
// Eij += sg (M_ij - conj(M_ji)).  (D = A - A^dagger is linear in A; reading R3.)
template <typename T>
__device__ __forceinline__ void acc_ah(const cx<T> (&m)[9], T sg, T (&di)[3], cx<T> (&E)[3])
{
    di[0] += sg * m[0].y; di[1] += sg * m[4].y; di[2] += sg * m[8].y;
    E[0].x += sg * (m[1].x - m[3].x); E[0].y += sg * (m[1].y + m[3].y);
    E[1].x += sg * (m[2].x - m[6].x); E[1].y += sg * (m[2].y + m[6].y);
    E[2].x += sg * (m[5].x - m[7].x); E[2].y += sg * (m[5].y + m[7].y);
}

// Delta = D - (1/3) Tr D with D = A - A^dagger given as di = Im A_ii and E = (D01, D02, D12):
// theta's Tr Delta Delta^dagger and the store of Delta in the packed (4) or full (9) field layout.
template <typename T, int PACK>
__device__ __forceinline__ double store_delta(const T (&di)[3], const cx<T> (&E)[3], cx<T> *__restrict__ wout, int64_t V, int64_t s)
{
    T d0 = 2 * di[0], d1 = 2 * di[1], d2 = 2 * di[2];
    const T m = (d0 + d1 + d2) * (T)(1.0 / 3.0);
    d0 -= m; d1 -= m; d2 -= m;
    const double th = (double)(d0 * d0 + d1 * d1 + d2 * d2) + 2.0 * (double)(cnorm2(E[0]) + cnorm2(E[1]) + cnorm2(E[2]));
    if (PACK == 4) {
        st_field(wout + s, mk<T>(d0, d1));
        st_field(wout + V + s, E[0]);
        st_field(wout + 2 * V + s, E[1]);
        st_field(wout + 3 * V + s, E[2]);
    } else {
        wout[s] = mk<T>(0, d0);
        wout[V + s] = E[0];
        wout[2 * V + s] = E[1];
        wout[3 * V + s] = mk<T>(-E[0].x, E[0].y);
        wout[4 * V + s] = mk<T>(0, d1);
        wout[5 * V + s] = E[2];
        wout[6 * V + s] = mk<T>(-E[1].x, E[1].y);
        wout[7 * V + s] = mk<T>(-E[2].x, E[2].y);
        wout[8 * V + s] = mk<T>(0, d2);
    }
    return th;
}

// STORE = false (LGF_OPT_ACCUM_G): `lin` holds the links as loaded, which stay where they are, and
// `gsrc` the accumulated transformation G(x) (rows 0, 1, updated by the last FFT pass).  The current
// links G(x) U_mu(x) G^dagger(x+mu) (Alg. 1 lines 12-16 applied n times) are formed in
// registers exactly as below and measured, but not written: 544 instead of 928 bytes per site
// (FP64, 12-real).
// ACCUM_G tuning (measured on B200, profiles/r01d_accum_g.md): with 18-real links the forward links
// are taken through their sum (rows 0, 1 of U suffice: 6 of 9 loads) at 3 CTAs per SM in FP64; with 12-real
// links the per-link form below at 4 CTAs per SM is faster (the sum form spills at 128 registers).
#ifndef LGF_ACC_QSUM
#define LGF_ACC_QSUM(NE) ((NE) == 9)
#endif
#ifndef LGF_ACC_MINB
#define LGF_ACC_MINB(NE, T) ((NE) == 9 && sizeof(T) == 8 ? 3 : 4)
#endif
// MARCH (LGF_OPT_TMARCH > 1): the thread walks tk consecutive time slices; a separate instantiation, so that the
// one-site form keeps its registers.
template <typename T, int NE, int PACK, bool GBUF, bool STORE, bool MARCH = false>
__global__ void __launch_bounds__(FUSED_THREADS, (STORE ? LGF_FUSED_MINB : LGF_ACC_MINB(NE, T)))
k_update_measure(const cx<T> *__restrict__ lin, cx<T> *__restrict__ lout, const cx<T> *__restrict__ gsrc,
                 cx<T> *__restrict__ wout, Geom geo, T a, int gexp, Ctrl *ctrl, double *partials, void *gred, double2 *hist, double eps, int tk_arg)
{
    const int tk = MARCH ? tk_arg : 1;
    if (*(volatile int *)&ctrl->done) return;
    const int64_t V = geo.V;
    const int64_t rr = (int64_t)blockIdx.x * FUSED_THREADS + threadIdx.x;
    double trF = 0, th = 0;
    if (rr < geo.Vw / tk) {
        int c[4];
        int64_t s = walk_site(geo, rr, c, tk);       // (z,t)-blocked walk: neighbour re-reads stay in L2
        if (!STORE && LGF_ACC_QSUM(NE)) {
            // ACCUM_G: nothing is stored, so the forward links enter only through their sum as well,
            //     sum_mu U'_mu(x) = G(x) [sum_mu U_mu(x) G^dagger(x+mu)]:
            // rows 0, 1 of U_mu(x) suffice (no third-row rebuild), G(x) is applied once.  The forward
            // bracket goes first so that G(x) is not live across both loops (registers).
            T di[3] = {0, 0, 0};
            cx<T> E[3] = {mk<T>(0, 0), mk<T>(0, 0), mk<T>(0, 0)};
            cx<T> X[9];
#pragma unroll
            for (int k = 0; k < 9; k++) X[k] = mk<T>(0, 0);
#pragma unroll
            for (int mu = 0; mu < 4; mu++) {
                const int64_t sp = s + (c[mu] == geo.N[mu] - 1 ? -(int64_t)(geo.N[mu] - 1) : (int64_t)1) * geo.st[mu];
                cx<T> g1[9], u[9], h[9];
                load_g01<T, PACK, GBUF>(gsrc, V, sp, a, gexp, g1);
                su3_row2(g1);
                const cx<T> *p = lin + (int64_t)mu * NE * V + s;
#pragma unroll
                for (int k = 0; k < 6; k++) u[k] = ld_link(p + (int64_t)k * V);
                mul_rows_dag<2>(u, g1, h);
                su3_row2(h);
#pragma unroll
                for (int k = 0; k < 9; k++) X[k] = X[k] + h[k];
            }
            {
                cx<T> g0[9], B[9];
                load_g01<T, PACK, GBUF>(gsrc, V, s, a, gexp, g0);
                su3_row2(g0);
                mul_rows<3>(g0, X, B);
                acc_ah<T>(B, (T)-1, di, E);
                trF = (double)(B[0].x + B[4].x + B[8].x);
            }
#pragma unroll
            for (int k = 0; k < 9; k++) X[k] = mk<T>(0, 0);
#pragma unroll
            for (int nu = 0; nu < 4; nu++) {
                const int64_t sb = s + (c[nu] == 0 ? (int64_t)(geo.N[nu] - 1) : (int64_t)-1) * geo.st[nu];
                cx<T> gb[9], u[9], h[9];
                load_g01<T, PACK, GBUF>(gsrc, V, sb, a, gexp, gb);
                load_link_in<T, NE>(lin, V, nu, sb, u);
                mul_rows<2>(gb, u, h);
                su3_row2(h);
#pragma unroll
                for (int k = 0; k < 9; k++) X[k] = X[k] + h[k];
            }
            {
                cx<T> g0[9], B[9];
                load_g01<T, PACK, GBUF>(gsrc, V, s, a, gexp, g0);   // again: an L1 hit, cheaper than 36 live registers
                su3_row2(g0);
                mul_rows_dag<3>(X, g0, B);
                acc_ah<T>(B, (T)1, di, E);
            }
            th = store_delta<T, PACK>(di, E, wout, V, s);
        } else {
#if LGF_FUSED_PREFETCH
            // The thread's own links are first touched by the forward products at the end of its life (a DRAM
            // round trip each); ask L2 for them now, behind the backward products.
#pragma unroll
            for (int k = 0; k < 4 * NE; k++) asm volatile("prefetch.global.L2 [%0];" ::"l"(lin + (int64_t)k * V + s));
#endif
            // LGF_OPT_TMARCH: the thread walks tk consecutive time slices.  The -t neighbour of its second, third ...
            // site is its own previous site, whose H_t = g U_t it has just formed for the forward product
            // (Tc below): 12 loads and one product less per site after the first.
            cx<T> Tc[6];
          for (int kk = 0; kk < tk; kk++) {
            // Backward links first: only their sum enters A'(x),
            //     sum_nu U'_nu(x-nu) = [sum_nu H_nu(x-nu)] g^dagger(x),   H_nu(y) = g(y) U_nu(y),
            // so rows 0, 1 of each H are one product, row 2 is conj(row0 x row1) (H is special
            // unitary) and g^dagger(x) is applied once to the sum.
            cx<T> X[9];
#pragma unroll
            for (int k = 0; k < 9; k++) X[k] = mk<T>(0, 0);
#pragma unroll
            for (int q = 0; q < 4; q++) {
                const int nu = LGF_FUSED_BWD_REV ? 3 - q : q;
                const int64_t sb = s + (c[nu] == 0 ? (int64_t)(geo.N[nu] - 1) : (int64_t)-1) * geo.st[nu];
                cx<T> h[9];
                if (MARCH && nu == 3 && kk > 0) {
#pragma unroll
                    for (int k = 0; k < 6; k++) h[k] = Tc[k];
#ifdef LGF_FUSED_SKIP_BWD   /* timing-only ceiling experiment (bit mask of directions whose backward link is NOT rebuilt): WRONG results */
                } else if ((LGF_FUSED_SKIP_BWD >> nu) & 1) {
#pragma unroll
                    for (int k = 0; k < 6; k++) h[k] = mk<T>(0, 0);
#endif
                } else {
                    cx<T> gb[9], u[9];
                    load_g01<T, PACK, GBUF>(gsrc, V, sb, a, gexp, gb);
                    load_link_in<T, NE>(lin, V, nu, sb, u);
                    mul_rows<2>(gb, u, h);
                }
                su3_row2(h);
#pragma unroll
                for (int k = 0; k < 9; k++) X[k] = X[k] + h[k];
            }
            cx<T> g0[9];
            load_g01<T, PACK, GBUF>(gsrc, V, s, a, gexp, g0);
            su3_row2(g0);
            T di[3] = {0, 0, 0};
            cx<T> E[3] = {mk<T>(0, 0), mk<T>(0, 0), mk<T>(0, 0)};
            {
                cx<T> B[9];
                mul_rows_dag<3>(X, g0, B);
                acc_ah<T>(B, (T)1, di, E);
            }
            // Forward links U'_mu(x) = g(x) U_mu(x) g^dagger(x+mu): rows 0, 1 computed and stored; row 2 is
            // conj(row0 x row1), which is also what a later load of 12-real storage rebuilds (R15).
            T tr = 0;
#pragma unroll
            for (int mu = 0; mu < 4; mu++) {
                const int64_t sp = s + (c[mu] == geo.N[mu] - 1 ? -(int64_t)(geo.N[mu] - 1) : (int64_t)1) * geo.st[mu];
                cx<T> g1[9], u[9], t[9], r[9];
                load_g01<T, PACK, GBUF>(gsrc, V, sp, a, gexp, g1);
                su3_row2(g1);
#ifdef LGF_FUSED_FAKE_OWN   /* timing-only experiment: the thread's own links come from a cache-resident window (WRONG results) */
                load_link_in<T, NE>(lin, V, mu, s & (int64_t)(LGF_FUSED_FAKE_OWN - 1), u);
#else
                load_link_in<T, NE>(lin, V, mu, s, u);
#endif
                mul_rows<2>(g0, u, t);
                if (MARCH && mu == 3) {
#pragma unroll
                    for (int k = 0; k < 6; k++) Tc[k] = t[k];
                }
                mul_rows_dag<2>(t, g1, r);
                su3_row2(r);
                if (STORE) {
                    cx<T> *p = lout + (int64_t)mu * NE * V + s;
#pragma unroll
                    for (int k = 0; k < NE; k++) st_link(p + (int64_t)k * V, r[k]);
                }
                tr += r[0].x + r[4].x + r[8].x;
                acc_ah<T>(r, (T)-1, di, E);
            }
            trF += (double)tr;
            th += store_delta<T, PACK>(di, E, wout, V, s);
            s += geo.st[3];
            c[3] += 1;
          }
        }
    }
#if LGF_REDUCE_2L
    finish_measure_2l<FUSED_THREADS>(trF, th, geo.Vg, ctrl, partials, gred, hist, eps, 1);
#else
    finish_measure<FUSED_THREADS>(trF, th, geo.Vg, ctrl, partials, hist, eps, 1);
#endif
}

int fused_blocks(int64_t V) { return (int)((V + FUSED_THREADS - 1) / FUSED_THREADS); }

// ---------------------------------------------------------------- the link kernel on 4D tiles (LGF_OPT_LINK_TILE)
// A'(x) (eq. 1.5) needs the new link U'_nu(x-nu) only through its anti-Hermitian part: Delta is linear
// in A - A^dagger.  k_update_measure lets the thread of x rebuild all four backward links from the old ones
// (24 more loads and 30 more complex multiply-adds per direction).  Here a CTA owns an Nx x TDy x TDz x TDt tile of
// sites, one thread per site.  The thread of x forms its four forward links once (Alg. 1 lines 12-16,
// PAPER.md:98-106), stores them, and leaves the nine reals of the anti-Hermitian part of each (Im of the diagonal,
// M_ij - conj(M_ji) above it) in shared memory; after one barrier the thread of x+nu picks them up.  Only the
// backward neighbours outside the tile (the tile faces; none along a direction the tile spans completely, where
// the neighbour wraps inside the tile) are rebuilt as before.  Same links as k_update_measure bit for bit; Delta,
// F, theta differ in the order of their sums only.
// MEASURED SLOWER on B200 (profiles/r02_link_tile.md: 32^4 FP64 12-real 238-261 us against 200 us, 64^4 5.18 against
// 4.21 ms, 48^4 FP32 994 against 660 us) and therefore off by default: the backward rebuilds it removes are L1 / L2
// hits that cost the site kernel only 7 % (LGF_FUSED_SKIP_BWD ceiling: 185.7 us), while the barrier in the middle of
// a CTA's life and the spills of the FP64 form cost more.  Kept so that the comparison can be re-run.
struct LinkTile {
    int TD[4];       // tile extents (TD[0] = Nx)
    int nT[4];       // tiles per direction
    int tv;          // sites per tile (<= threads per CTA)
    int zbt;         // z-block of the tile walk, in tiles (divides nT[2])
};

// the nine reals of the anti-Hermitian part of one link
template <typename T> __device__ __forceinline__ void ah_part(const cx<T> (&m)[9], T (&p)[9])
{
    p[0] = m[0].y; p[1] = m[4].y; p[2] = m[8].y;
    p[3] = m[1].x - m[3].x; p[4] = m[1].y + m[3].y;
    p[5] = m[2].x - m[6].x; p[6] = m[2].y + m[6].y;
    p[7] = m[5].x - m[7].x; p[8] = m[5].y + m[7].y;
}

template <typename T, int NE, int PACK, bool GBUF, int THREADS>
__global__ void __launch_bounds__(THREADS, 512 / THREADS)
k_update_measure_tile(const cx<T> *__restrict__ lin, cx<T> *__restrict__ lout, const cx<T> *__restrict__ gsrc,
                      cx<T> *__restrict__ wout, Geom geo, LinkTile tg, T a, int gexp, Ctrl *ctrl, double *partials, double2 *hist, double eps)
{
    if (*(volatile int *)&ctrl->done) return;
    extern __shared__ __align__(16) unsigned char xs_raw[];
    T *xs = (T *)xs_raw;                             // [direction][9][THREADS]
    const int64_t V = geo.V;
    const int l = threadIdx.x;
    const bool active = l < tg.tv;
    // tile of this CTA: y-tiles fastest, then the (z,t) tiles in z-blocks like walk_site
    unsigned b = blockIdx.x;
    const int ty = (int)(b % (unsigned)tg.nT[1]); b /= (unsigned)tg.nT[1];
    const unsigned per = (unsigned)(tg.zbt * tg.nT[3]);
    const unsigned zblk = b / per, rem = b % per;
    const int tt = (int)(rem / (unsigned)tg.zbt), tz = (int)(zblk * (unsigned)tg.zbt + rem % (unsigned)tg.zbt);
    int lc[4], c[4];
    {
        unsigned r = (unsigned)l;
        lc[0] = (int)(r % (unsigned)tg.TD[0]); r /= (unsigned)tg.TD[0];
        lc[1] = (int)(r % (unsigned)tg.TD[1]); r /= (unsigned)tg.TD[1];
        lc[2] = (int)(r % (unsigned)tg.TD[2]); r /= (unsigned)tg.TD[2];
        lc[3] = (int)r;
    }
    c[0] = lc[0]; c[1] = ty * tg.TD[1] + lc[1]; c[2] = tz * tg.TD[2] + lc[2]; c[3] = tt * tg.TD[3] + lc[3];
    const int64_t s = c[0] + geo.st[1] * c[1] + geo.st[2] * c[2] + geo.st[3] * c[3];
    int lst[4];                                      // thread-index stride of each direction inside the tile
    lst[0] = 1; lst[1] = tg.TD[0]; lst[2] = tg.TD[0] * tg.TD[1]; lst[3] = tg.TD[0] * tg.TD[1] * tg.TD[2];
    double trF = 0, th = 0;
    if (active) {
        cx<T> g0[9];
        load_g01<T, PACK, GBUF>(gsrc, V, s, a, gexp, g0);
        su3_row2(g0);
        T tr = 0;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const int64_t sp = s + (c[mu] == geo.N[mu] - 1 ? -(int64_t)(geo.N[mu] - 1) : (int64_t)1) * geo.st[mu];
            cx<T> g1[9], u[9], t[9], r[9];
            load_g01<T, PACK, GBUF>(gsrc, V, sp, a, gexp, g1);
            su3_row2(g1);
            load_link_in<T, NE>(lin, V, mu, s, u);
            mul_rows<2>(g0, u, t);
            mul_rows_dag<2>(t, g1, r);
            su3_row2(r);
            cx<T> *p = lout + (int64_t)mu * NE * V + s;
#pragma unroll
            for (int k = 0; k < NE; k++) st_link(p + (int64_t)k * V, r[k]);
            tr += r[0].x + r[4].x + r[8].x;
            // the thread's own share of A'(x), -U'_mu(x), is read back from shared memory as well: nine accumulators
            // less to keep across the four products
            T q[9];
            ah_part<T>(r, q);
#pragma unroll
            for (int k = 0; k < 9; k++) xs[(mu * 9 + k) * THREADS + l] = q[k];
        }
        trF = (double)tr;
    }
    __syncthreads();
    if (active) {
        T D[9];
#pragma unroll
        for (int k = 0; k < 9; k++) D[k] = -((xs[k * THREADS + l] + xs[(9 + k) * THREADS + l]) + (xs[(18 + k) * THREADS + l] + xs[(27 + k) * THREADS + l]));
        cx<T> X[9];
#pragma unroll
        for (int k = 0; k < 9; k++) X[k] = mk<T>(0, 0);
        bool halo = false;
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const int nu = LGF_FUSED_BWD_REV ? 3 - q : q;
            if (tg.TD[nu] > 1 && (lc[nu] > 0 || tg.nT[nu] == 1)) {       // the neighbour is a thread of this CTA
                const int nl = l + (lc[nu] > 0 ? -1 : tg.TD[nu] - 1) * lst[nu];
#pragma unroll
                for (int k = 0; k < 9; k++) D[k] += xs[(nu * 9 + k) * THREADS + nl];
            } else {
                const int64_t sb = s + (c[nu] == 0 ? (int64_t)(geo.N[nu] - 1) : (int64_t)-1) * geo.st[nu];
                cx<T> gb[9], u[9], h[9];
                load_g01<T, PACK, GBUF>(gsrc, V, sb, a, gexp, gb);
                load_link_in<T, NE>(lin, V, nu, sb, u);
                mul_rows<2>(gb, u, h);
                su3_row2(h);
#pragma unroll
                for (int k = 0; k < 9; k++) X[k] = X[k] + h[k];
                halo = true;
            }
        }
        if (halo) {
            cx<T> g0[9], B[9];
            load_g01<T, PACK, GBUF>(gsrc, V, s, a, gexp, g0);    // again: an L1 hit, cheaper than 36 live registers
            su3_row2(g0);
            mul_rows_dag<3>(X, g0, B);
            T q[9];
            ah_part<T>(B, q);
#pragma unroll
            for (int k = 0; k < 9; k++) D[k] += q[k];
        }
        const T di[3] = {D[0], D[1], D[2]};
        const cx<T> E[3] = {mk<T>(D[3], D[4]), mk<T>(D[5], D[6]), mk<T>(D[7], D[8])};
        th = store_delta<T, PACK>(di, E, wout, V, s);
    }
    finish_measure<THREADS>(trF, th, geo.Vg, ctrl, partials, hist, eps, 1);
}

static void link_tile_set(const Geom &g, const int td[4], LinkTile &tg)
{
    for (int d = 0; d < 4; d++) { tg.TD[d] = td[d]; tg.nT[d] = g.N[d] / td[d]; }
    tg.tv = td[0] * td[1] * td[2] * td[3];
    // z-block of the walk in tiles: the site walk's block if it is a whole number of tiles
    const int zbt = g.zb / tg.TD[2];
    tg.zbt = (zbt >= 1 && g.zb % tg.TD[2] == 0 && tg.nT[2] % zbt == 0) ? zbt : tg.nT[2];
}

// Tile of `threads` sites at most: TD0 = Nx, the other extents divisors of Ny, Nz, Nt chosen to minimise the share of
// rebuilt backward links, sum_nu [TD_nu < N_nu] / TD_nu, weighted against idle threads.  Returns false when Nx > threads.
// Built with -DLGF_TILE_ENV the environment variable LGF_LINK_TILE_DIMS="TDy,TDz,TDt" overrides the choice (tuning sweeps).
static bool link_tile_choose(const Geom &g, int threads, LinkTile &tg)
{
    if (g.N[0] > threads) return false;
#ifdef LGF_TILE_ENV
    if (const char *e = getenv("LGF_LINK_TILE_DIMS")) {
        int a1, a2, a3;
        if (sscanf(e, "%d,%d,%d", &a1, &a2, &a3) == 3 && a1 > 0 && a2 > 0 && a3 > 0 && g.N[0] * a1 * a2 * a3 <= threads &&
            g.N[1] % a1 == 0 && g.N[2] % a2 == 0 && g.N[3] % a3 == 0) {
            const int td[4] = {g.N[0], a1, a2, a3};
            link_tile_set(g, td, tg);
            return true;
        }
    }
#endif
    double best = 1e30;
    int bt[4] = {g.N[0], 1, 1, 1};
    for (int a1 = 1; a1 <= g.N[1]; a1++) if (g.N[1] % a1 == 0)
        for (int a2 = 1; a2 <= g.N[2]; a2++) if (g.N[2] % a2 == 0)
            for (int a3 = 1; a3 <= g.N[3]; a3++) if (g.N[3] % a3 == 0) {
                const int tv = g.N[0] * a1 * a2 * a3;
                if (tv > threads) continue;
                const int td[4] = {g.N[0], a1, a2, a3};
                double halo = 0;
                for (int d = 1; d < 4; d++) halo += td[d] == g.N[d] ? 0.0 : 1.0 / td[d];
                const double cost = (1.0 + 0.3 * halo) * (double)threads / tv;
                if (cost < best - 1e-12) { best = cost; for (int d = 0; d < 4; d++) bt[d] = td[d]; }
            }
    link_tile_set(g, bt, tg);
    return true;
}

int link_tile_threads(const Geom &g, int want)
{
    LinkTile tg;
    if (g.Vw != g.V) return 0;                       // sharded slabs (halo slices, no wrap in t) keep the site kernel
    if (want != 128 && want != 256 && want != 512) return 0;
    if (!link_tile_choose(g, want, tg)) return 0;
    // one pair of partial sums per CTA: the workspace holds 2 fused_blocks(V) + 2 pairs (make_layout)
    return (int64_t)tg.nT[1] * tg.nT[2] * tg.nT[3] <= 2 * (int64_t)fused_blocks(g.V) ? want : 0;
}

template <typename T, int NE, int PACK, bool GB, int THREADS>
static void launch_tile_one(const SiteArgs &a, const LinkTile &tg, const void *lin, void *lout, const void *gsrc, void *wout,
                            double alpha, double eps, cudaStream_t st)
{
    const size_t smem = (size_t)4 * 9 * THREADS * sizeof(T);
    static bool done = false;
    if (!done) {
        done = true;
        if (cudaFuncSetAttribute(k_update_measure_tile<T, NE, PACK, GB, THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            cudaGetLastError();
    }
    const unsigned nb = (unsigned)(tg.nT[1] * tg.nT[2] * tg.nT[3]);
    k_update_measure_tile<T, NE, PACK, GB, THREADS><<<nb, THREADS, smem, st>>>((const cx<T> *)lin, (cx<T> *)lout, (const cx<T> *)gsrc,
        (cx<T> *)wout, a.geo, tg, (T)(alpha / 2.0), a.gexp, a.ctrl, a.partials, a.hist, eps);
}

static void launch_update_measure_tile(const SiteArgs &a, const void *lin, void *lout, const void *gsrc, int gbuf, void *wout,
                                       double alpha, double eps, cudaStream_t st)
{
    LinkTile tg;
    link_tile_choose(a.geo, a.ltile, tg);
#define CALL_T(T, NE, PACK, GB)                                                                                   \
    do {                                                                                                          \
        if (a.ltile == 128) launch_tile_one<T, NE, PACK, GB, 128>(a, tg, lin, lout, gsrc, wout, alpha, eps, st);  \
        else if (a.ltile == 256) launch_tile_one<T, NE, PACK, GB, 256>(a, tg, lin, lout, gsrc, wout, alpha, eps, st); \
        else launch_tile_one<T, NE, PACK, GB, 512>(a, tg, lin, lout, gsrc, wout, alpha, eps, st);                 \
    } while (0)
#define CALL_NE(T, NE)                                           \
    do {                                                         \
        if (gbuf) { CALL_T(T, NE, 4, true); }                    \
        else if (a.pack == 4) { CALL_T(T, NE, 4, false); }       \
        else { CALL_T(T, NE, 9, false); }                        \
    } while (0)
    if (a.prec == 0) { if (a.recon == 12) CALL_NE(double, 6); else CALL_NE(double, 9); }
    else             { if (a.recon == 12) CALL_NE(float, 6); else CALL_NE(float, 9); }
#undef CALL_NE
#undef CALL_T
}

// ---------------------------------------------------------------- the link kernel as a stream (LGF_OPT_LINK_STREAM)
// The same arithmetic as k_update_measure, site by site, with the thread's OWN links -- the 4 NE lines per site that
// must come from DRAM -- fetched ahead of time by the TMA engine instead of by the thread: a persistent CTA walks
// tiles of TS consecutive sites of the walk order (contiguous in memory when Nx Ny is a multiple of TS); its producer
// warp issues one cp.async.bulk per SoA component array (TS x 16 bytes, contiguous) into a ring of shared-memory
// stages, completion on an mbarrier, and the consumer warps take U_mu(x) -- and U_nu(x-nu) where x-nu lies in the
// tile -- from shared memory.  g and the backward links outside the tile come through L1 / L2 as before.  Bytes in
// flight per SM are then set by the ring (stages x 4 NE x TS x 16 B), not by the registers of 16 warps.
// F and theta are accumulated per thread over all tiles of the CTA and reduced once at the end (one pair of partial
// sums per CTA), so they differ from the site kernel's in the order of the sums only; links bitwise equal.
// Default path only (g buffer, 4 packed fields); lattices with Nx Ny % TS != 0 and sharded slabs keep the site kernel.
#ifndef LGF_STREAM_STAGES
#define LGF_STREAM_STAGES 2
#endif
#ifdef LGF_STREAM_MINB_ALL   /* tuning sweeps: one CTA count for every instantiation (nvcc splits -D values at commas) */
#define LGF_STREAM_MINB(T, NE) LGF_STREAM_MINB_ALL
#endif
#ifndef LGF_STREAM_MINB
#define LGF_STREAM_MINB(T, NE) ((sizeof(T) == 8 && (NE) == 9) ? 1 : 2)
#endif
static const int STREAM_TS = 128;                    // sites per tile = consumer threads
static const int STREAM_THREADS = STREAM_TS + 32;    // + one producer warp

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *b, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *b, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *b)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned long long *b, unsigned parity)
{
    unsigned ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(unsigned long long *b, unsigned parity)
{
    while (!mbar_try_wait(b, parity)) {}
}
// global -> shared bulk copy by the TMA engine (UBLKCP in SASS); bytes: multiple of 16, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

template <typename T, int NE> struct StreamCfg {
    static constexpr int NARR = 4 * NE;
    static constexpr size_t STAGE = (size_t)NARR * STREAM_TS * sizeof(cx<T>);
    static constexpr int NST = LGF_STREAM_STAGES;
    static constexpr size_t SMEM = 128 + (size_t)NST * STAGE;     // barriers in the first 128 bytes
    static constexpr int MINB = LGF_STREAM_MINB(T, NE);
};

// U_mu of site index s: from the stage when s lies in the tile [s0, s0 + TS), else from global memory
template <typename T, int NE>
__device__ __forceinline__ void load_link_stream(const cx<T> *__restrict__ lin, const cx<T> *stg, int64_t V, int mu, int64_t s, int64_t s0, cx<T> (&u)[9])
{
    const int64_t d = s - s0;
    if ((unsigned long long)d < (unsigned long long)STREAM_TS) {
        const cx<T> *p = stg + (size_t)mu * NE * STREAM_TS + d;
#pragma unroll
        for (int k = 0; k < NE; k++) u[k] = p[k * STREAM_TS];
        if (NE == 6) su3_row2(u);
    } else {
        load_link_in<T, NE>(lin, V, mu, s, u);
    }
}

template <typename T, int NE>
__global__ void __launch_bounds__(STREAM_THREADS, (StreamCfg<T, NE>::MINB))
k_update_measure_stream(const cx<T> *__restrict__ lin, cx<T> *__restrict__ lout, const cx<T> *__restrict__ gsrc,
                        cx<T> *__restrict__ wout, Geom geo, int ntiles, Ctrl *ctrl, double *partials, double2 *hist, double eps)
{
    if (*(volatile int *)&ctrl->done) return;
    typedef StreamCfg<T, NE> CF;
    constexpr int TS = STREAM_TS, NST = CF::NST;
    extern __shared__ __align__(128) unsigned char st_raw[];
    unsigned long long *full = (unsigned long long *)st_raw, *empty = full + NST;
    cx<T> *stage0 = (cx<T> *)(st_raw + 128);
    const int tid = threadIdx.x;
    const int64_t V = geo.V;
    if (tid == 0) {
        for (int i = 0; i < NST; i++) { mbar_init(full + i, 1); mbar_init(empty + i, TS / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    double trF = 0, th = 0;
    if (tid >= TS) {
        // ---- producer warp: lane 0 keeps the ring full, the other lanes walk along (the warp stays converged)
        int st = 0;
        unsigned ph = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            if (tid == TS) {
                mbar_wait(empty + st, ph ^ 1u);                        // the consumers are done with this stage
                int c[4];
                const int64_t s0 = walk_site(geo, (int64_t)tile * TS, c);
                cx<T> *dst = stage0 + (size_t)st * CF::NARR * TS;
                mbar_expect_tx(full + st, (unsigned)CF::STAGE);
#pragma unroll 4
                for (int j = 0; j < CF::NARR; j++)
                    bulk_g2s(dst + (size_t)j * TS, lin + (int64_t)j * V + s0, (unsigned)(TS * sizeof(cx<T>)), full + st);
            }
            __syncwarp();
            if (++st == NST) { st = 0; ph ^= 1u; }
        }
    } else {
        // ---- consumers: one site per thread and tile
        int st = 0;
        unsigned ph = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            int c[4];
            const int64_t s = walk_site(geo, (int64_t)tile * TS + tid, c);
            const int64_t s0 = s - tid;
            const cx<T> *stg = stage0 + (size_t)st * CF::NARR * TS;
            // backward links, order t, z, y, x: t and z lie in other planes (global memory, issued before the wait);
            // y and x are in the tile for most sites
            cx<T> X[9];
#pragma unroll
            for (int k = 0; k < 9; k++) X[k] = mk<T>(0, 0);
#pragma unroll
            for (int q = 0; q < 4; q++) {
                const int nu = 3 - q;
                const int64_t sb = s + (c[nu] == 0 ? (int64_t)(geo.N[nu] - 1) : (int64_t)-1) * geo.st[nu];
                cx<T> gb[9], u[9], h[9];
                load_g01<T, 4, true>(gsrc, V, sb, (T)0, 0, gb);
                if (nu >= 2) {
                    load_link_in<T, NE>(lin, V, nu, sb, u);
                } else {
                    if (nu == 1) mbar_wait(full + st, ph);             // the tile's own links have landed
                    load_link_stream<T, NE>(lin, stg, V, nu, sb, s0, u);
                }
                mul_rows<2>(gb, u, h);
                su3_row2(h);
#pragma unroll
                for (int k = 0; k < 9; k++) X[k] = X[k] + h[k];
            }
            cx<T> g0[9];
            load_g01<T, 4, true>(gsrc, V, s, (T)0, 0, g0);
            su3_row2(g0);
            T di[3] = {0, 0, 0};
            cx<T> E[3] = {mk<T>(0, 0), mk<T>(0, 0), mk<T>(0, 0)};
            {
                cx<T> B[9];
                mul_rows_dag<3>(X, g0, B);
                acc_ah<T>(B, (T)1, di, E);
            }
            T tr = 0;
#pragma unroll
            for (int mu = 0; mu < 4; mu++) {
                const int64_t sp = s + (c[mu] == geo.N[mu] - 1 ? -(int64_t)(geo.N[mu] - 1) : (int64_t)1) * geo.st[mu];
                cx<T> g1[9], u[9], t[9], r[9];
                load_g01<T, 4, true>(gsrc, V, sp, (T)0, 0, g1);
                su3_row2(g1);
                {
                    const cx<T> *p = stg + (size_t)mu * NE * TS + tid;
#pragma unroll
                    for (int k = 0; k < NE; k++) u[k] = p[k * TS];
                    if (NE == 6) su3_row2(u);
                }
                if (mu == 3) {                                         // last read of the stage: hand it back
                    __syncwarp();
                    if ((tid & 31) == 0) mbar_arrive(empty + st);
                }
                mul_rows<2>(g0, u, t);
                mul_rows_dag<2>(t, g1, r);
                su3_row2(r);
                cx<T> *p = lout + (int64_t)mu * NE * V + s;
#pragma unroll
                for (int k = 0; k < NE; k++) st_link(p + (int64_t)k * V, r[k]);
                tr += r[0].x + r[4].x + r[8].x;
                acc_ah<T>(r, (T)-1, di, E);
            }
            trF += (double)tr;
            th += store_delta<T, 4>(di, E, wout, V, s);
            if (++st == NST) { st = 0; ph ^= 1u; }
        }
    }
    finish_measure<STREAM_THREADS>(trF, th, geo.Vg, ctrl, partials, hist, eps, 1);
}

// 1 when the streamed link kernel applies to this geometry
int link_stream_ok(const Geom &g)
{
    if (g.Vw != g.V) return 0;                                    // sharded slabs keep the site kernel
    return ((int64_t)g.N[0] * g.N[1]) % STREAM_TS == 0 ? 1 : 0;
}

template <typename T, int NE>
static void launch_stream_one(const SiteArgs &a, const void *lin, void *lout, const void *gsrc, void *wout, double eps, cudaStream_t st)
{
    typedef StreamCfg<T, NE> CF;
    static int resident = 0;
    if (resident == 0) {
        int dev = 0, sms = 148, per = 1;
        if (cudaFuncSetAttribute(k_update_measure_stream<T, NE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CF::SMEM) != cudaSuccess) cudaGetLastError();
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); sms = 148; }
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k_update_measure_stream<T, NE>, STREAM_THREADS, CF::SMEM) != cudaSuccess || per < 1) { cudaGetLastError(); per = 1; }
        resident = sms * per;
    }
    const int ntiles = (int)(a.geo.V / STREAM_TS);
    const int nb = ntiles < resident ? ntiles : resident;
    k_update_measure_stream<T, NE><<<nb, STREAM_THREADS, CF::SMEM, st>>>((const cx<T> *)lin, (cx<T> *)lout, (const cx<T> *)gsrc, (cx<T> *)wout,
        a.geo, ntiles, a.ctrl, a.partials, a.hist, eps);
}

static void launch_update_measure_stream(const SiteArgs &a, const void *lin, void *lout, const void *gsrc, void *wout, double eps, cudaStream_t st)
{
    if (a.prec == 0) { if (a.recon == 12) launch_stream_one<double, 6>(a, lin, lout, gsrc, wout, eps, st); else launch_stream_one<double, 9>(a, lin, lout, gsrc, wout, eps, st); }
    else             { if (a.recon == 12) launch_stream_one<float, 6>(a, lin, lout, gsrc, wout, eps, st); else launch_stream_one<float, 9>(a, lin, lout, gsrc, wout, eps, st); }
}

// The link kernel keeps nothing in shared memory but the reduction scratch: ask for the largest L1
// the SM offers, the x and y neighbours of a CTA's sites are re-read through it (once per instantiation).
#ifndef LGF_FUSED_MAXL1
#define LGF_FUSED_MAXL1 1
#endif
template <typename T, int NE, int PACK, bool GBUF, bool STORE> static void prefer_l1()
{
#if LGF_FUSED_MAXL1
    static bool done = false;
    if (done) return;
    done = true;
    if (cudaFuncSetAttribute(k_update_measure<T, NE, PACK, GBUF, STORE, false>, cudaFuncAttributePreferredSharedMemoryCarveout,
                             (int)cudaSharedmemCarveoutMaxL1) != cudaSuccess)
        cudaGetLastError();
    if (cudaFuncSetAttribute(k_update_measure<T, NE, PACK, GBUF, STORE, true>, cudaFuncAttributePreferredSharedMemoryCarveout,
                             (int)cudaSharedmemCarveoutMaxL1) != cudaSuccess)
        cudaGetLastError();
#endif
}

void launch_update_measure(const SiteArgs &a, const void *lin, void *lout, const void *gsrc, int gbuf, void *wout,
                           double alpha, double eps, cudaStream_t st)
{
    if (a.lstream > 0 && gbuf) { launch_update_measure_stream(a, lin, lout, gsrc, wout, eps, st); return; }
    if (a.ltile > 0) { launch_update_measure_tile(a, lin, lout, gsrc, gbuf, wout, alpha, eps, st); return; }
    const int tk = a.tmarch > 0 ? a.tmarch : 1;
    const int nb = fused_blocks(a.geo.Vw / tk);
#define CALL(T, NE, PACK, GB) \
    do { prefer_l1<T, NE, PACK, GB, true>();   \
    if (tk > 1) k_update_measure<T, NE, PACK, GB, true, true><<<nb, FUSED_THREADS, LGF_FUSED_DUMMY_SMEM, st>>>((const cx<T> *)lin, (cx<T> *)lout, (const cx<T> *)gsrc, \
        (cx<T> *)wout, a.geo, (T)(alpha / 2.0), a.gexp, a.ctrl, a.partials, a.gred, a.hist, eps, tk); \
    else k_update_measure<T, NE, PACK, GB, true, false><<<nb, FUSED_THREADS, LGF_FUSED_DUMMY_SMEM, st>>>((const cx<T> *)lin, (cx<T> *)lout, (const cx<T> *)gsrc, \
        (cx<T> *)wout, a.geo, (T)(alpha / 2.0), a.gexp, a.ctrl, a.partials, a.gred, a.hist, eps, 1); } while (0)
#define CALL_NE(T, NE)                                           \
    do {                                                         \
        if (gbuf) { CALL(T, NE, 4, true); }                      \
        else if (a.pack == 4) { CALL(T, NE, 4, false); }         \
        else { CALL(T, NE, 9, false); }                          \
    } while (0)
    if (a.prec == 0) { if (a.recon == 12) CALL_NE(double, 6); else CALL_NE(double, 9); }
    else             { if (a.recon == 12) CALL_NE(float, 6); else CALL_NE(float, 9); }
#undef CALL_NE
#undef CALL
}

void launch_measure_acc(const SiteArgs &a, const void *gacc, double eps, cudaStream_t st)
{
    // the 18-real form sums the forward links first (LGF_ACC_QSUM) and walks one site per thread
    const int tk = (a.tmarch > 0 && !(LGF_ACC_QSUM(a.recon == 12 ? 6 : 9))) ? a.tmarch : 1;
    const int nb = fused_blocks(a.geo.Vw / tk);
#define CALL(T, NE) \
    do { prefer_l1<T, NE, 4, true, false>();  \
    if (tk > 1) k_update_measure<T, NE, 4, true, false, true><<<nb, FUSED_THREADS, 0, st>>>((const cx<T> *)a.links, (cx<T> *)nullptr, \
        (const cx<T> *)gacc, (cx<T> *)a.w, a.geo, (T)0, 0, a.ctrl, a.partials, a.gred, a.hist, eps, tk); \
    else k_update_measure<T, NE, 4, true, false, false><<<nb, FUSED_THREADS, 0, st>>>((const cx<T> *)a.links, (cx<T> *)nullptr, \
        (const cx<T> *)gacc, (cx<T> *)a.w, a.geo, (T)0, 0, a.ctrl, a.partials, a.gred, a.hist, eps, 1); } while (0)
    if (a.prec == 0) { if (a.recon == 12) CALL(double, 6); else CALL(double, 9); }
    else             { if (a.recon == 12) CALL(float, 6); else CALL(float, 9); }
#undef CALL
}

} // namespace lgf
