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
#include "launch.h"
#include "twiddles.cuh"
#include "su3.cuh"
#include <cooperative_groups.h>

namespace lgf {

// ---------------------------------------------------------------- twiddles
// exp(SIGN 2 pi i k / L) from the literal tables; L divides 64 or 48.
template <typename T, int L, int SIGN> __device__ __forceinline__ cx<T> twiddle(int k)
{
    constexpr bool b64 = (64 % L == 0);
    constexpr int B = b64 ? 64 : 48;
    static_assert(B % L == 0, "line length must divide 64 or 48");
    const int i = (k % L) * (B / L);
    const double c = b64 ? TW_COS64[b64 ? i : 0] : TW_COS48[b64 ? 0 : i];
    const double s = b64 ? TW_SIN64[b64 ? i : 0] : TW_SIN48[b64 ? 0 : i];
    return mk<T>((T)c, (T)(SIGN * s));
}

// x * exp(SIGN 2 pi i k / L), trivial factors resolved at compile time (k is known after unrolling)
template <typename T, int L, int SIGN> __device__ __forceinline__ cx<T> mul_tw(cx<T> x, int k)
{
    k %= L;
    if (k == 0) return x;
    if (2 * k == L) return mk<T>(-x.x, -x.y);
    if (4 * k == L) return SIGN > 0 ? mk<T>(-x.y, x.x) : mk<T>(x.y, -x.x);       // * (+-i)
    if (4 * k == 3 * L) return SIGN > 0 ? mk<T>(x.y, -x.x) : mk<T>(-x.y, x.x);   // * (-+i)
    return cmul(x, twiddle<T, L, SIGN>(k));
}

// ---------------------------------------------------------------- radix-p butterflies
template <typename T, int SIGN> __device__ __forceinline__ void bfly3(cx<T> &a0, cx<T> &a1, cx<T> &a2)
{
    const T h = (T)0.86602540378443865; // sqrt(3)/2
    const cx<T> t1 = a1 + a2;
    const cx<T> t2 = mk<T>(a0.x - (T)0.5 * t1.x, a0.y - (T)0.5 * t1.y);
    const cx<T> d = a1 - a2;
    // SIGN * i * h * d
    const cx<T> t3 = SIGN > 0 ? mk<T>(-h * d.y, h * d.x) : mk<T>(h * d.y, -h * d.x);
    a0 = a0 + t1;
    a1 = t2 + t3;
    a2 = t2 - t3;
}

// One decimation-in-frequency stage on blocks of length L (L = p m): butterfly over the p
// sub-blocks, then multiply sub-block q by exp(SIGN 2 pi i j q / L); recurse on length m.
template <typename T, int N, int L, int SIGN> struct Dif {
    static __device__ __forceinline__ void run(cx<T> (&x)[N])
    {
        constexpr int p = (L % 2 == 0) ? 2 : 3;
        constexpr int m = L / p;
#pragma unroll
        for (int b = 0; b < N; b += L)
#pragma unroll
            for (int j = 0; j < m; j++) {
                if (p == 2) {
                    const cx<T> a = x[b + j], c = x[b + j + m];
                    x[b + j] = a + c;
                    x[b + j + m] = mul_tw<T, L, SIGN>(a - c, j);
                } else {
                    bfly3<T, SIGN>(x[b + j], x[b + j + m], x[b + j + 2 * m]);
                    x[b + j + m] = mul_tw<T, L, SIGN>(x[b + j + m], j);
                    x[b + j + 2 * m] = mul_tw<T, L, SIGN>(x[b + j + 2 * m], 2 * j);
                }
            }
        Dif<T, N, m, SIGN>::run(x);
    }
};
template <typename T, int N, int SIGN> struct Dif<T, N, 1, SIGN> {
    static __device__ __forceinline__ void run(cx<T> (&)[N]) {}
};

// The transposed network: stages in the opposite order, twiddles before the butterfly.
// Takes the slot order Dif produces and returns natural order.
template <typename T, int N, int L, int SIGN> struct Dit {
    static __device__ __forceinline__ void run(cx<T> (&x)[N])
    {
        constexpr int p = (L % 2 == 0) ? 2 : 3;
        constexpr int m = L / p;
        Dit<T, N, m, SIGN>::run(x);
#pragma unroll
        for (int b = 0; b < N; b += L)
#pragma unroll
            for (int j = 0; j < m; j++) {
                if (p == 2) {
                    const cx<T> a = x[b + j], c = mul_tw<T, L, SIGN>(x[b + j + m], j);
                    x[b + j] = a + c;
                    x[b + j + m] = a - c;
                } else {
                    x[b + j + m] = mul_tw<T, L, SIGN>(x[b + j + m], j);
                    x[b + j + 2 * m] = mul_tw<T, L, SIGN>(x[b + j + 2 * m], 2 * j);
                    bfly3<T, SIGN>(x[b + j], x[b + j + m], x[b + j + 2 * m]);
                }
            }
    }
};
template <typename T, int N, int SIGN> struct Dit<T, N, 1, SIGN> {
    static __device__ __forceinline__ void run(cx<T> (&)[N]) {}
};

// frequency index held by slot s after Dif<N> (mixed-radix digit reversal)
template <int N> __host__ __device__ constexpr int slot_freq(int s)
{
    int L = N, k = 0, mult = 1;
    while (L > 1) {
        const int p = (L % 2 == 0) ? 2 : 3, m = L / p;
        k += (s / m) * mult;
        s %= m;
        mult *= p;
        L = m;
    }
    return k;
}

// ---------------------------------------------------------------- a line held by S threads
// S = 1: one thread holds the whole line.  S = 2: the line is shared by the lanes l and l^16 of
// a warp (half h = 0, 1).  The first radix-2 stage of the decimation-in-frequency network,
//     y[j] = x[j] + x[j+N/2],   z[j] = (x[j] - x[j+N/2]) exp(SIGN 2 pi i j/N),   j < N/2,
// is done on the pairs each thread holds (j in [h N/4, (h+1) N/4)); then the two threads swap
// half of their results by warp shuffle so that h = 0 owns all of y (even frequencies) and
// h = 1 all of z (odd frequencies), and each runs the N/2-point network on its own.
// The transposed (decimation-in-time) network runs the same steps backwards.
// nat(i, h): line position held in local element i on the natural-order side;
// slot(s, h): frequency (or position, for an inverse written as Dif) held in local slot s on the other side.
template <typename T, int N, int S> struct Line;

template <typename T, int N> struct Line<T, N, 1> {
    static constexpr int NL = N;
    static __device__ __forceinline__ int nat(int i, int) { return i; }
    static __device__ __forceinline__ int slot(int s, int) { return slot_freq<N>(s); }
    template <int SIGN> static __device__ __forceinline__ void dif(cx<T> (&v)[NL], int, unsigned) { Dif<T, N, N, SIGN>::run(v); }
    template <int SIGN> static __device__ __forceinline__ void dit(cx<T> (&v)[NL], int, unsigned) { Dit<T, N, N, SIGN>::run(v); }
};

template <typename V> __device__ __forceinline__ V shfl16(unsigned mask, V v)
{
    v.x = __shfl_xor_sync(mask, v.x, 16);
    v.y = __shfl_xor_sync(mask, v.y, 16);
    return v;
}
// x * (SIGN i)
template <int SIGN, typename V> __device__ __forceinline__ V rot90(V x)
{
    V r;
    if (SIGN > 0) { r.x = -x.y; r.y = x.x; } else { r.x = x.y; r.y = -x.x; }
    return r;
}

template <typename T, int N> struct Line<T, N, 2> {
    static_assert(N % 4 == 0, "split lines need N divisible by 4");
    static constexpr int NL = N / 2, Q = N / 4;
    static __device__ __forceinline__ int nat(int i, int h) { return h * Q + i + (i >= Q ? Q : 0); }
    static __device__ __forceinline__ int slot(int s, int h) { return 2 * slot_freq<NL>(s) + h; }
    template <int SIGN> static __device__ __forceinline__ void dif(cx<T> (&v)[NL], int h, unsigned mask)
    {
#pragma unroll
        for (int i = 0; i < Q; i++) {
            const cx<T> a = v[i], b = v[Q + i];
            const cx<T> y = a + b;
            cx<T> z = mul_tw<T, N, SIGN>(a - b, i);
            if (h) z = rot90<SIGN>(z);                       // exp(SIGN 2 pi i (N/4)/N) = SIGN i
            const cx<T> got = shfl16(mask, h ? y : z);       // h = 0 gives z away, h = 1 gives y away
            v[i] = h ? got : y;
            v[Q + i] = h ? z : got;
        }
        Dif<T, NL, NL, SIGN>::run(v);
    }
    template <int SIGN> static __device__ __forceinline__ void dit(cx<T> (&v)[NL], int h, unsigned mask)
    {
        Dit<T, NL, NL, SIGN>::run(v);
#pragma unroll
        for (int i = 0; i < Q; i++) {
            const cx<T> got = shfl16(mask, h ? v[i] : v[Q + i]);
            const cx<T> y = h ? got : v[i];
            cx<T> z = h ? v[Q + i] : got;
            z = mul_tw<T, N, SIGN>(z, i);
            if (h) z = rot90<SIGN>(z);
            v[i] = y + z;
            v[Q + i] = y - z;
        }
    }
};

// thread t of a group -> (line, half).  S = 2 keeps the two halves of a line 16 lanes apart, so
// that the 8 lanes of a shared-memory wavefront still belong to 8 consecutive lines.
template <int S> __device__ __forceinline__ void line_of_thread(int t, int &line, int &h)
{
    if (S == 1) { line = t; h = 0; }
    else { h = (t >> 4) & 1; line = (t & 15) | ((t >> 5) << 4); }
}
// Lines of at least SMIN points are shared by two lanes.  48 and 64 must be (registers).  32-point
// lines are split for FP64 tiles with NA == NB only: a same-run A/B at 32^4 FP64 gave 0.3164 against
// 0.3279 ms per iteration (twice the warps per tile at 84-128 instead of 146-196 registers), while FP32
// tiles and the (32, 48) / (32, 64) (z,t) tiles of 32^3 x n lattices got 5-15 % slower
// (profiles/r01e_final.md).  LGF_SPLIT_MIN overrides the rule for tuning sweeps.
#ifdef LGF_SPLIT_MIN
template <typename T> constexpr int split_min(int, int) { return LGF_SPLIT_MIN; }
#else
template <typename T> constexpr int split_min(int na, int nb) { return (sizeof(T) == 8 && na == nb) ? 32 : 48; }
#endif
constexpr int split_of(int n, int smin) { return n >= smin ? 2 : 1; }

// ---------------------------------------------------------------- tile geometry
// Shared tile of a group: element (c, a, b) at (b*RS + a*C + c), RS = NA*C + C (one padding
// column block per row keeps 16-byte accesses of 8 consecutive threads on distinct banks).
// Lines along a: C*NB of them, SA threads each; lines along b: C*NA, SB threads each.
constexpr int imax(int a, int b) { return a > b ? a : b; }
template <int NA, int NB, int C, int SMIN> struct Tile {
    static constexpr int SA = split_of(NA, SMIN), SB = split_of(NB, SMIN);
    static constexpr int RS = NA * C + C;
    static constexpr int ELEMS = RS * NB;
    static constexpr int THREADS = C * imax(SA * NB, SB * NA);
};
// CTA size: at least 128 threads, whole groups
constexpr int cta_threads(int group) { return group >= 128 ? group : (128 / group) * group; }

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

template <typename T, int NA, int NB, int INVERSE>
__global__ void __launch_bounds__((XYCfg<T, NA, NB>::CTA))
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
// 266 KB): a thread-block CLUSTER of two CTAs holds the plane, two fields each; after the
// transforms each CTA builds g for half of the sites, reading its own two fields locally and
// the other two from the peer's shared memory (DSMEM).
template <typename T, int NA, int NB> struct XYG2Cfg {
    typedef Tile<NA, NB, 1, split_min<T>(NA, NB)> TL;
    static constexpr int TP = (TL::SA > 1 || TL::SB > 1) ? (TL::THREADS + 31) / 32 * 32 : TL::THREADS;
    static constexpr int CTA = 2 * TP;                        // two fields per CTA
    static constexpr size_t SMEM = (size_t)2 * TL::ELEMS * sizeof(cx<T>);
    static constexpr bool FITS = SMEM <= 227 * 1024 && CTA <= 1024 && CTA >= 64;
};

template <typename T, int NA, int NB, bool ACC>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__((XYG2Cfg<T, NA, NB>::CTA))
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
    const int rank = (int)cluster.block_rank();              // 0: fields 0, 1;  1: fields 2, 3
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T> *smp = (cx<T> *)smem_raw;
    const int t = threadIdx.x, lf = t / TP, l = t % TP;
    cx<T> *sm = smp + (size_t)lf * TL::ELEMS;
    const int64_t plane = blockIdx.x >> 1;
    const int64_t base = plane * (int64_t)(NA * NB);
    int xa, ha, yb, hb;
    line_of_thread<TL::SB>(l, xa, ha);
    line_of_thread<TL::SA>(l, yb, hb);
    const bool on_y = xa < NA && l < TL::SB * NA, on_x = yb < NB && l < TL::SA * NB;
    const unsigned my = __ballot_sync(0xffffffffu, on_y), mx = __ballot_sync(0xffffffffu, on_x);
    {
        const cx<T> *f = w + (int64_t)(2 * rank + lf) * V + base;
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
    const cx<T> *peer = cluster.map_shared_rank(smp, rank ^ 1);
    const cx<T> *f01 = rank == 0 ? smp : peer, *f23 = rank == 0 ? peer : smp;
    constexpr int HALF = NA * NB / 2;
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
                m_from_packed<T>(f01[o], f01[TL::ELEMS + o], f23[o], f23[TL::ELEMS + o], a, g);
                finish_g01<T>(g, gexp);
                emit_g<T, ACC>(g, Gold[b], gbuf + base + i, V);
            }
        }
    }
    cluster.sync();                                          // the peer may still be reading this CTA's fields
}

// ---------------------------------------------------------------- pass 1: (z,t) tiles
// Tile = C consecutive x at fixed (field, y): element (c, z, t) at global x0 + c + sz*z + st*t.
// z-lines straight from global (thread = (c, t)), Dif(-) along z -> shared; t-lines from
// shared (thread = (c, kz)): Dif(-), mask, Dit(+) -> shared; z-lines from shared: Dif(+),
// stored straight to global.  p^2 = sum_mu 4 sin^2(pi k_mu/N_mu) (reading R5) from the
// per-axis tables; the factor p_max^2/(p^2 V) is one FP64 division per mode.
#ifndef LGF_ZT_MAXB
#define LGF_ZT_MAXB 2   /* 3 measured slower at 32^4 (47.6 vs 45.5 us: spills), equal at 48^4 */
#endif
template <typename T, int NA, int NB, int C> struct ZTCfg {
    typedef Tile<NA, NB, C, split_min<T>(NA, NB)> TL;
    static constexpr int TT = TL::THREADS;
    static constexpr int CTA = cta_threads(TT);
    static constexpr int G = CTA / TT;
    static constexpr size_t PT = ((NB * sizeof(double) + 15) / 16) * 16;
    static constexpr size_t SMEM = PT + (size_t)G * TL::ELEMS * sizeof(cx<T>);
    // CTAs per SM that shared memory allows (1 KB reserved each); registers are capped to match
    static constexpr int FIT = (int)((size_t)227 * 1024 / (SMEM + 1024));
    static constexpr int MINB = FIT < 1 ? 1 : (FIT > LGF_ZT_MAXB ? LGF_ZT_MAXB : FIT);
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
        for (int i = 0; i < LA::NL; i++) v[i] = g[sz * LA::nat(i, ha)];
        LA::template dif<-1>(v, ha, mz);
#pragma unroll
        for (int q = 0; q < LA::NL; q++) sm[ta * TL::RS + LA::slot(q, ha) * C + ca] = v[q];
    }
    __syncthreads();
    if (on_t) {                                                        // t-line at (c, kz) = (cb, zb)
        cx<T> v[LB::NL];
#pragma unroll
        for (int i = 0; i < LB::NL; i++) v[i] = sm[LB::nat(i, hb) * TL::RS + zb * C + cb];
        LB::template dif<-1>(v, hb, mt);
        const double pxyz = ptab[x0 + cb] + ptab[Nx + y] + ptab[Nx + Ny + zb];
#pragma unroll
        for (int q = 0; q < LB::NL; q++) {
            const double p2 = pxyz + pt[LB::slot(q, hb)];
            const T fac = (p2 > 0.0) ? (T)(pmax2_over_V / p2) : (T)0;  // zero mode -> 0 (reading R7)
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
        for (int i = 0; i < LA::NL; i++) v[i] = sm[ta * TL::RS + LA::nat(i, ha) * C + ca];
        LA::template dif<+1>(v, ha, mz);
        cx<T> *g = f + ca + st * ta;
#pragma unroll
        for (int q = 0; q < LA::NL; q++) g[sz * LA::slot(q, ha)] = v[q];
    }
}

// ---------------------------------------------------------------- dispatch
// x-columns per (z,t) tile: 64-byte runs in global memory (FP64), unless the tile would not fit
#ifndef LGF_ZT_BYTES
#define LGF_ZT_BYTES 64
#endif
template <typename T, int NA, int NB> struct ZTC {
    static constexpr int WANT = LGF_ZT_BYTES / (int)sizeof(cx<T>);
    static constexpr size_t tile_bytes(int c) { return (size_t)(NA * c + c) * NB * sizeof(cx<T>); }
    static constexpr int C = tile_bytes(WANT) <= 200 * 1024 && NA % WANT == 0 ? WANT : (tile_bytes(WANT / 2) <= 200 * 1024 && NA % (WANT / 2) == 0 ? WANT / 2 : WANT / 4);
};

template <typename T, int N> static int setup_xy_n()
{
    cudaError_t e;
    e = cudaFuncSetAttribute(k_fft_xy<T, N, N, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYCfg<T, N, N>::SMEM);
    if (e != cudaSuccess) return 1;
    e = cudaFuncSetAttribute(k_fft_xy<T, N, N, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYCfg<T, N, N>::SMEM);
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

template <typename T, int NA, int NB> static int setup_zt_n()
{
    constexpr int C = ZTC<T, NA, NB>::C;
    typedef ZTCfg<T, NA, NB, C> Z;
    cudaError_t e = cudaFuncSetAttribute(k_fft_zt<T, NA, NB, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Z::SMEM);
    return e == cudaSuccess ? 0 : 1;
}

template <typename T, int NA, int NB> static int launch_zt_n(const FftArgs &a, cudaStream_t st)
{
    constexpr int C = ZTC<T, NA, NB>::C;
    typedef ZTCfg<T, NA, NB, C> Z;
    const int64_t ntiles = (int64_t)a.nfields * a.geo.N[1] * (a.geo.N[0] / C);
    const unsigned grid = (unsigned)((ntiles + Z::G - 1) / Z::G);
    k_fft_zt<T, NA, NB, C><<<grid, Z::CTA, Z::SMEM, st>>>((cx<T> *)a.w, a.geo, a.ptab, a.pmax2 / (double)a.geo.V, ntiles, a.ctrl);
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
        if (accum) k_fft_xy_inv_g2<T, N, N, true><<<(unsigned)(2 * nplanes), X::CTA, X::SMEM, st>>>((const cx<T> *)a.w, (cx<T> *)gbuf, a.geo.V, (T)(alpha / 2.0), gexp, a.ctrl);
        else k_fft_xy_inv_g2<T, N, N, false><<<(unsigned)(2 * nplanes), X::CTA, X::SMEM, st>>>((const cx<T> *)a.w, (cx<T> *)gbuf, a.geo.V, (T)(alpha / 2.0), gexp, a.ctrl);
    }
    return 0;
}

template <typename T, int N> static int gbuf_fits_n() { return (XYGCfg<T, N, N>::FITS || XYG2Cfg<T, N, N>::FITS) ? 1 : 0; }

// Lattices with Nx = Ny in {8, 12, 16, 24, 32, 48, 64} and (Nz, Nt) either equal and in the same
// set or (32, n), n in {8, 16, 48, 64} (the paper's 32^3 x n lattices): the (x,y)
// passes are instantiated per Nx and the (z,t) pass per (Nz, Nt).  The x-columns of a (z,t) tile
// must divide Nx (2 or 4).  Everything else takes the generic path.
static bool tiled_extent(int n) { return n == 8 || n == 16 || n == 32 || n == 64 || n == 12 || n == 24 || n == 48; }
static bool tiled_zt(int nz, int nt)
{
    if (nz == nt) return tiled_extent(nz);
    return nz == 32 && (nt == 8 || nt == 16 || nt == 48 || nt == 64);
}
bool fft_tiled_supported(const int N[4], int prec)
{
    (void)prec;
    return N[0] == N[1] && tiled_extent(N[0]) && tiled_zt(N[2], N[3]);
}

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
// (z,t) pass: FN<T, Nz, Nt> for the supported pairs
#define LGF_ZT_CASE(FN, A, B, ...) \
    if (nz == A && nt == B) return prec == 0 ? FN<double, A, B>(__VA_ARGS__) : FN<float, A, B>(__VA_ARGS__);
#define LGF_ZT_SWITCH(FN, ...)                                                                              \
    LGF_ZT_CASE(FN, 8, 8, __VA_ARGS__) LGF_ZT_CASE(FN, 12, 12, __VA_ARGS__) LGF_ZT_CASE(FN, 16, 16, __VA_ARGS__) \
    LGF_ZT_CASE(FN, 24, 24, __VA_ARGS__) LGF_ZT_CASE(FN, 32, 32, __VA_ARGS__) LGF_ZT_CASE(FN, 48, 48, __VA_ARGS__) \
    LGF_ZT_CASE(FN, 64, 64, __VA_ARGS__) LGF_ZT_CASE(FN, 32, 8, __VA_ARGS__) LGF_ZT_CASE(FN, 32, 16, __VA_ARGS__) \
    LGF_ZT_CASE(FN, 32, 48, __VA_ARGS__) LGF_ZT_CASE(FN, 32, 64, __VA_ARGS__)

static int setup_zt(int nz, int nt, int prec)
{
    LGF_ZT_SWITCH(setup_zt_n)
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
    const int nz = a.geo.N[2], nt = a.geo.N[3], prec = a.prec;
    LGF_ZT_SWITCH(launch_zt_n, a, st)
    return 1;
}
void launch_fft_tiled(const FftArgs &a, int which, cudaStream_t st)
{
    if (which == 1) run_zt(a, st); else run_xy(a, which, st);
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
