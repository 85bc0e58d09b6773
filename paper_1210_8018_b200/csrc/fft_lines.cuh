// fft_lines.cuh -- the 1D transforms of the tiled FFT (Alg. 1 lines 3-8): a whole
// line held in the registers of one thread, or of two lanes of a warp, transformed by a fully
// unrolled decimation-in-frequency network with compile-time twiddles.  Shared by the (x,y) passes
// (fft_tiled.cu) and the (z,t) pass (fft_zt.cuh); see the header of fft_tiled.cu for the pass structure.
#pragma once
#include "launch.h"
#include "twiddles.cuh"

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

// S = 4: the line is shared by the four lanes l, l^8, l^16, l^24 of a warp, quarter h = 2 a + b (a: lane bit 4,
// b: lane bit 3), N/4 elements each: the two-lane scheme applied twice.  Lane h starts with the positions
// [h N/8, (h+1) N/8) and the same plus N/2; the first radix-2 stage and an exchange across bit a leave y
// (even frequencies) in the lanes a = 0 and z (odd) in a = 1, each N/2-point sequence shared by the two lanes b = 0, 1
// exactly as a two-lane line is; the second stage and an exchange across bit b leave every lane with an
// N/4-point sequence of its own.  Slot s of lane (a, b) ends up holding frequency 4 slot_freq<N/4>(s) + a + 2 b.
// Same number of shuffles and selects per thread as the two-lane form of a line of half the length, half the
// registers per thread and twice the threads per line: for kernels that are bound by latency at 16 warps per
// SM (profiles/r02_fft_passes.md).
template <typename V> __device__ __forceinline__ V shfl8(unsigned mask, V v)
{
    v.x = __shfl_xor_sync(mask, v.x, 8);
    v.y = __shfl_xor_sync(mask, v.y, 8);
    return v;
}
template <typename T, int N> struct Line<T, N, 4> {
    static_assert(N % 8 == 0, "four-lane lines need N divisible by 8");
    static constexpr int NL = N / 4, Q = N / 8, M = N / 2;
    static __device__ __forceinline__ int nat(int i, int h) { return h * Q + (i >= Q ? i - Q + M : i); }
    static __device__ __forceinline__ int slot(int s, int h) { return 4 * slot_freq<NL>(s) + (h >> 1) + 2 * (h & 1); }
    // exp(SIGN 2 pi i h / 8): the part of the first-stage twiddle exp(SIGN 2 pi i (h Q + i) / N) that depends on the lane
    template <int SIGN> static __device__ __forceinline__ cx<T> lane_tw(int h)
    {
        const T r = (T)0.70710678118654752440;
        const T re = h == 0 ? (T)1 : (h == 1 ? r : (h == 2 ? (T)0 : -r));
        const T im = h == 0 ? (T)0 : (h == 2 ? (T)1 : r);
        return mk<T>(re, SIGN > 0 ? im : -im);
    }
    template <int SIGN> static __device__ __forceinline__ void dif(cx<T> (&v)[NL], int h, unsigned mask)
    {
        const int a = h >> 1, b = h & 1;
        const cx<T> lt = lane_tw<SIGN>(h);
#pragma unroll
        for (int i = 0; i < Q; i++) {                        // stage 1 on N points, exchange across bit a
            const cx<T> p = v[i], q = v[Q + i];
            const cx<T> y = p + q;
            const cx<T> z = cmul(mul_tw<T, N, SIGN>(p - q, i), lt);
            const cx<T> got = shfl16(mask, a ? y : z);
            v[i] = a ? got : y;
            v[Q + i] = a ? z : got;
        }
#pragma unroll
        for (int i = 0; i < Q; i++) {                        // stage 2 on N/2 points, exchange across bit b
            const cx<T> p = v[i], q = v[Q + i];
            const cx<T> y = p + q;
            cx<T> z = mul_tw<T, M, SIGN>(p - q, i);
            if (b) z = rot90<SIGN>(z);
            const cx<T> got = shfl8(mask, b ? y : z);
            v[i] = b ? got : y;
            v[Q + i] = b ? z : got;
        }
        Dif<T, NL, NL, SIGN>::run(v);
    }
    template <int SIGN> static __device__ __forceinline__ void dit(cx<T> (&v)[NL], int h, unsigned mask)
    {
        const int a = h >> 1, b = h & 1;
        const cx<T> lt = lane_tw<SIGN>(h);
        Dit<T, NL, NL, SIGN>::run(v);
#pragma unroll
        for (int i = 0; i < Q; i++) {
            const cx<T> got = shfl8(mask, b ? v[i] : v[Q + i]);
            const cx<T> y = b ? got : v[i];
            cx<T> z = b ? v[Q + i] : got;
            z = mul_tw<T, M, SIGN>(z, i);
            if (b) z = rot90<SIGN>(z);
            v[i] = y + z;
            v[Q + i] = y - z;
        }
#pragma unroll
        for (int i = 0; i < Q; i++) {
            const cx<T> got = shfl16(mask, a ? v[i] : v[Q + i]);
            const cx<T> y = a ? got : v[i];
            cx<T> z = a ? v[Q + i] : got;
            z = cmul(mul_tw<T, N, SIGN>(z, i), lt);
            v[i] = y + z;
            v[Q + i] = y - z;
        }
    }
};

// thread t of a group -> (line, part).  S = 2 keeps the two halves of a line 16 lanes apart (S = 4: the four
// quarters 8 lanes apart), so that the 8 lanes of a shared-memory wavefront still belong to 8 consecutive lines.
template <int S> __device__ __forceinline__ void line_of_thread(int t, int &line, int &h)
{
    if (S == 1) { line = t; h = 0; }
    else if (S == 2) { h = (t >> 4) & 1; line = (t & 15) | ((t >> 5) << 4); }
    else { h = (t >> 3) & 3; line = (t & 7) | ((t >> 5) << 3); }
}
// Lines of at least SMIN points are shared by two lanes.  48 and 64 must be (registers).  32-point
// lines are split for FP64 tiles with NA == NB only: a same-run A/B at 32^4 FP64 gave 0.3164 against
// 0.3279 ms per iteration (twice the warps per tile at 84-128 instead of 146-196 registers), while FP32
// tiles and the (32, 48) / (32, 64) (z,t) tiles of 32^3 x n lattices got 5-15 % slower
// (profiles/r01e_final.md).  LGF_SPLIT_MIN overrides the rule for tuning sweeps.
// LGF_SPLIT4_MIN: lines of at least that many points are shared by four lanes (FP64 tiles with NA == NB only; 0 = never).
#ifndef LGF_SPLIT4_MIN
#define LGF_SPLIT4_MIN 0
#endif
#ifdef LGF_SPLIT_MIN
template <typename T> constexpr int split_min2(int, int) { return LGF_SPLIT_MIN; }
#else
template <typename T> constexpr int split_min2(int na, int nb) { return (sizeof(T) == 8 && na == nb) ? 32 : 48; }
#endif
// the two thresholds packed into one template argument: (four-lane threshold << 8) | two-lane threshold
template <typename T> constexpr int split_min(int na, int nb)
{
    return ((sizeof(T) == 8 && na == nb && LGF_SPLIT4_MIN > 0 ? LGF_SPLIT4_MIN : 255) << 8) | split_min2<T>(na, nb);
}
constexpr int split_of(int n, int smin) { return n >= (smin >> 8) ? 4 : (n >= (smin & 255) ? 2 : 1); }

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

// p_max^2 / (p^2 V) for one mode (eq. 1.2; zero mode -> 0, reading R7): c = p_max^2 / V.
// The reciprocal is the hardware seed (MUFU.RCP64H, about 20 bits) refined by two Newton steps, each
// of which doubles the number of correct bits: p^2 is a sum of four numbers in [0, 4], so none of the
// special cases of an IEEE division can occur and its slow path (a CALL per mode in SASS: 16 per thread
// and tile, a sixth of the FP64 instructions of this pass) is dead weight.  Result within 2 ulp of c / p2.
__device__ __forceinline__ double mask_factor(double c, double p2)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(p2));
    double e = fma(-p2, y, 1.0);
    y = fma(y, e, y);
    e = fma(-p2, y, 1.0);
    y = fma(y, e, y);
    return (p2 > 0.0) ? c * y : 0.0;
}


} // namespace lgf
