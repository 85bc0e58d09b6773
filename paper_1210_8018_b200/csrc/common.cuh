// common.cuh -- shared device-side types of liblgf (CUDA path only; shares nothing with oracle/).
//
// Notation follows arXiv 1210.8018: V sites, N_c = 3, links U_mu(x), Delta(x) (eq. 1.5),
// F (eq. 1.1), theta (eq. 1.4).  Site index s = ix + Nx*(iy + Ny*(iz + Nz*it)).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lgf {

// ---------------------------------------------------------------- complex numbers
template <typename T> struct C2;
template <> struct C2<double> { typedef double2 type; };
template <> struct C2<float> { typedef float2 type; };
template <typename T> using cx = typename C2<T>::type;

template <typename T> __host__ __device__ __forceinline__ cx<T> mk(T re, T im) { cx<T> r; r.x = re; r.y = im; return r; }
__device__ __forceinline__ double2 operator+(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 operator-(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
// Complex products written as explicit fused multiply-adds: `acc.x += a.x*b.x - a.y*b.y` as plain
// C++ costs DMUL + DFMA + DADD per component (the compiler may not reassociate), the forms
// below cost two FMAs.  The FP64 pipe is the second roofline of this path.
__device__ __forceinline__ double fma_t(double a, double b, double c) { return ::fma(a, b, c); }
__device__ __forceinline__ float fma_t(float a, float b, float c) { return ::fmaf(a, b, c); }
// a*b
template <typename V> __device__ __forceinline__ V cmul(V a, V b)
{
    V r;
    r.x = fma_t(-a.y, b.y, a.x * b.x);
    r.y = fma_t(a.y, b.x, a.x * b.y);
    return r;
}
// a*conj(b)
template <typename V> __device__ __forceinline__ V cmulc(V a, V b)
{
    V r;
    r.x = fma_t(a.y, b.y, a.x * b.x);
    r.y = fma_t(-a.x, b.y, a.y * b.x);
    return r;
}
// conj(a)*b
template <typename V> __device__ __forceinline__ V cconjmul(V a, V b)
{
    V r;
    r.x = fma_t(a.y, b.y, a.x * b.x);
    r.y = fma_t(-a.y, b.x, a.x * b.y);
    return r;
}
// acc + a*b
template <typename V> __device__ __forceinline__ V cfma(V a, V b, V acc)
{
    acc.x = fma_t(-a.y, b.y, fma_t(a.x, b.x, acc.x));
    acc.y = fma_t(a.y, b.x, fma_t(a.x, b.y, acc.y));
    return acc;
}
// acc - a*b
template <typename V> __device__ __forceinline__ V cfms(V a, V b, V acc)
{
    acc.x = fma_t(a.y, b.y, fma_t(-a.x, b.x, acc.x));
    acc.y = fma_t(-a.y, b.x, fma_t(-a.x, b.y, acc.y));
    return acc;
}
// acc + a*conj(b)
template <typename V> __device__ __forceinline__ V cfmac(V a, V b, V acc)
{
    acc.x = fma_t(a.y, b.y, fma_t(a.x, b.x, acc.x));
    acc.y = fma_t(-a.x, b.y, fma_t(a.y, b.x, acc.y));
    return acc;
}
// acc + conj(a)*b
template <typename V> __device__ __forceinline__ V cfmaconj(V a, V b, V acc)
{
    acc.x = fma_t(a.y, b.y, fma_t(a.x, b.x, acc.x));
    acc.y = fma_t(-a.y, b.x, fma_t(a.x, b.y, acc.y));
    return acc;
}
// ---------------------------------------------------------------- packed FP32 (sm_100: add / mul / fma .f32x2)
// A complex number in FP32 is a register pair, and Blackwell has arithmetic on pairs (FADD2, FMUL2, FFMA2 in SASS):
// a complex add is one instruction, a complex multiply-add two (the broadcasts {a.x, a.x} and the swaps {b.y, b.x}
// become operand modifiers).  Same operations as the scalar forms above up to which of the two products of a
// component is rounded first.  Measured on B200 (same-run A/B, profiles/r02_f32x2.md): 43 % fewer arithmetic
// instructions in the FP32 FFT passes but register-pair moves in their place; the (x,y) passes on 32^2 planes get
// 10-16 % faster, the 48^2 passes and the (z,t) pass do not change, the FP32 link kernel gets 8-9 % SLOWER.  So the
// packed forms are compiled in the translation unit of the (x,y) passes only (fft_tiled.cu defines LGF_F32X2 1 before
// it includes this header); -DLGF_F32X2=0 / 1 on the command line sets it everywhere.
#ifndef LGF_F32X2
#define LGF_F32X2 0
#endif
#if LGF_F32X2
__device__ __forceinline__ unsigned long long pk2(float lo, float hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float2 un2(unsigned long long r)
{
    float2 v;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(v.x), "=f"(v.y) : "l"(r));
    return v;
}
__device__ __forceinline__ unsigned long long mul2(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ float2 add2(float2 a, float2 b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a.x, a.y)), "l"(pk2(b.x, b.y)));
    return un2(r);
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b)
{
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a.x, a.y)), "l"(pk2(b.x, b.y)));
    return un2(r);
}
// non-template overloads: preferred over the templates above for float2
__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return un2(fma2(pk2(a.x, a.x), pk2(b.x, b.y), mul2(pk2(a.y, a.y), pk2(-b.y, b.x)))); }
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) { return un2(fma2(pk2(a.x, a.x), pk2(b.x, -b.y), mul2(pk2(a.y, a.y), pk2(b.y, b.x)))); }
__device__ __forceinline__ float2 cconjmul(float2 a, float2 b) { return un2(fma2(pk2(a.x, a.x), pk2(b.x, b.y), mul2(pk2(a.y, a.y), pk2(b.y, -b.x)))); }
__device__ __forceinline__ float2 cfma(float2 a, float2 b, float2 acc) { return un2(fma2(pk2(a.y, a.y), pk2(-b.y, b.x), fma2(pk2(a.x, a.x), pk2(b.x, b.y), pk2(acc.x, acc.y)))); }
__device__ __forceinline__ float2 cfms(float2 a, float2 b, float2 acc) { return un2(fma2(pk2(a.y, a.y), pk2(b.y, -b.x), fma2(pk2(-a.x, -a.x), pk2(b.x, b.y), pk2(acc.x, acc.y)))); }
__device__ __forceinline__ float2 cfmac(float2 a, float2 b, float2 acc) { return un2(fma2(pk2(a.y, a.y), pk2(b.y, b.x), fma2(pk2(a.x, a.x), pk2(b.x, -b.y), pk2(acc.x, acc.y)))); }
__device__ __forceinline__ float2 cfmaconj(float2 a, float2 b, float2 acc) { return un2(fma2(pk2(a.y, a.y), pk2(b.y, -b.x), fma2(pk2(a.x, a.x), pk2(b.x, b.y), pk2(acc.x, acc.y)))); }
__device__ __forceinline__ float2 cscale(float2 a, float s) { return un2(mul2(pk2(a.x, a.y), pk2(s, s))); }
#endif
#if LGF_F32X2
__device__ __forceinline__ float2 operator+(float2 a, float2 b) { return add2(a, b); }
__device__ __forceinline__ float2 operator-(float2 a, float2 b) { return sub2(a, b); }
#else
__device__ __forceinline__ float2 operator+(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 operator-(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
#endif
template <typename V> __device__ __forceinline__ V cconj(V a) { a.y = -a.y; return a; }
template <typename V> __device__ __forceinline__ auto cnorm2(V a) -> decltype(a.x) { return a.x * a.x + a.y * a.y; }
template <typename V, typename T> __device__ __forceinline__ V cscale(V a, T s) { a.x *= s; a.y *= s; return a; }

// ---------------------------------------------------------------- lattice geometry
struct Geom {
    int N[4];        // Nx, Ny, Nz, Nt
    int64_t V;       // sites
    int64_t st[4];   // site-index stride of each direction: 1, Nx, Nx*Ny, Nx*Ny*Nz
    int zb;          // z-block of the site walk (divides Nz; Nz = plain lexicographic order), see walk_site
    // One lattice sharded over several GPUs in t-slabs (LGF_OPT_SHARD_WORLD): the arrays of a
    // rank hold its Ntw time slices between one halo slice below and one above, N[3] = Ntw + 2, t0 = 1, so the
    // t-neighbours of a walked site never wrap; the per-site kernels walk the Vw interior sites only and
    // normalise F and theta by the Vg sites of the whole lattice.  Unsharded: Vw = Vg = V, Ntw = N[3], t0 = 0.
    int64_t Vw, Vg;
    int Ntw, t0;
};

__device__ __forceinline__ void site_coords(const Geom &g, int64_t s, int c[4])
{
    unsigned u = (unsigned)s;               // V <= 64^4 < 2^32: 32-bit divisions
    c[0] = (int)(u % (unsigned)g.N[0]); u /= (unsigned)g.N[0];
    c[1] = (int)(u % (unsigned)g.N[1]); u /= (unsigned)g.N[1];
    c[2] = (int)(u % (unsigned)g.N[2]); u /= (unsigned)g.N[2];
    c[3] = (int)u;
}

// Walk order of the per-site kernels: grid thread r (= blockIdx.x * blockDim.x + threadIdx.x) -> site.
// Inside one (z,t) plane the order is the storage order (x fastest), so warps still read contiguous
// runs.  The planes are visited in blocks of geo.zb consecutive z: all Nt time slices of one z-block
// before the next z-block,
//     r -> (o, q) = (r mod NxNy, r div NxNy),   q -> (zblk, t, zin),   z = zblk*zb + zin.
// CTAs that are resident together then cover neighbouring z AND neighbouring t: the -t and +t
// neighbours of a site are zb planes away in the walk instead of Nz planes, so that the re-reads of
// U_nu(x-nu), g(x-nu), g(x+mu) (Alg. 1 lines 12-16) are L2 hits even when one time
// slice of links is larger than L2 (64^4: 151 MB per slice).  Only the first
// plane of a z-block misses its -z neighbours (1/zb of the sites).  zb = Nz is the lexicographic order.
// Returns the site index and fills c[0..3]; valid for r < Vw.
// tk > 1 (the link kernel's LGF_OPT_TMARCH): a thread handles tk consecutive time slices; r then runs over Vw / tk
// threads and the site returned is the first of the tk.
__device__ __forceinline__ int64_t walk_site(const Geom &g, int64_t r, int c[4], int tk = 1)
{
    const unsigned P = (unsigned)(g.N[0] * g.N[1]);
    const unsigned u = (unsigned)r;          // V <= 64^4 = 2^24
    const unsigned o = u % P, q = u / P;
    c[0] = (int)(o % (unsigned)g.N[0]);
    c[1] = (int)(o / (unsigned)g.N[0]);
    const unsigned per = (unsigned)(g.zb * (g.Ntw / tk));
    const unsigned zblk = q / per, rem = q % per;
    c[3] = (int)(rem / (unsigned)g.zb) * tk + g.t0;
    c[2] = (int)(zblk * (unsigned)g.zb + rem % (unsigned)g.zb);
    return (int64_t)o + (int64_t)P * (c[2] + g.N[2] * c[3]);
}

// ---------------------------------------------------------------- device control block
// One per context, in the workspace.  The stop decision of Algorithm 1 is
// taken by the last block of kernel (a) and kept here, so that the host need not read
// theta back after every iteration.
#define LGF_HIST_CAP 4096   /* = LGF_HISTORY_CAP of include/lgf.h (static_assert in lgf_api.cu) */
struct Ctrl {
    double F;                 // eq. 1.1 of the current links
    double theta;             // eq. 1.4
    long long iter;           // loop-body executions since the last reset
    int done;                 // 0 running, 1 theta <= eps reached, 2 theta is NaN/Inf
    unsigned int ticket;      // block counter of the fixed-order final reduction
    int pad[2];
};

} // namespace lgf
