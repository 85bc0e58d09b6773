// su3.cuh -- 3x3 complex matrix helpers in registers (CUDA path only).
#pragma once
#include "common.cuh"

namespace lgf {

// Third row of a special unitary matrix from rows 0, 1: row2 = conj(row0 x row1)
// (12-real compression; reading R15).  m[0..5] given, m[6..8] written.
template <typename V> __device__ __forceinline__ void su3_row2(V (&m)[9])
{
    m[6] = cconj(cfms(m[2], m[4], cmul(m[1], m[5])));
    m[7] = cconj(cfms(m[0], m[5], cmul(m[2], m[3])));
    m[8] = cconj(cfms(m[1], m[3], cmul(m[0], m[4])));
}

// Load U_mu(s) from the SoA link arrays: element k = 3*row + col of direction mu lives at
// links[(mu*NE + k)*V + s], NE = 9 (18-real) or 6 (12-real, row 2 rebuilt here).
template <typename T, int NE>
__device__ __forceinline__ void load_link(const cx<T> *__restrict__ links, int64_t V, int mu, int64_t s, cx<T> (&u)[9])
{
    const cx<T> *p = links + (int64_t)mu * NE * V + s;
#pragma unroll
    for (int k = 0; k < NE; k++) u[k] = __ldg(p + (int64_t)k * V);
    if (NE == 6) su3_row2(u);
}

// The same through plain (coherent) loads, for the kernels that rewrite the link buffer in place (k_update,
// k_apply_g): ld.global.nc promises that the data is read-only for the whole kernel, which an in-place
// update does not honour even though every thread reads its own links before it writes them.
template <typename T, int NE>
__device__ __forceinline__ void load_link_rw(const cx<T> *links, int64_t V, int mu, int64_t s, cx<T> (&u)[9])
{
    const cx<T> *p = links + (int64_t)mu * NE * V + s;
#pragma unroll
    for (int k = 0; k < NE; k++) u[k] = p[(int64_t)k * V];
    if (NE == 6) su3_row2(u);
}

template <typename T> __device__ __forceinline__ T rsqrt_t(T x);
template <> __device__ __forceinline__ double rsqrt_t<double>(double x) { return rsqrt(x); }
template <> __device__ __forceinline__ float rsqrt_t<float>(float x) { return rsqrtf(x); }

// Gram-Schmidt on rows 0, 1 of m in place ("followed by a reunitarization";
// DESIGN.md readings R12, R13).  Row 2 is not touched.
template <typename T> __device__ __forceinline__ void reunit01(cx<T> (&g)[9])
{
    T n0 = rsqrt_t<T>(cnorm2(g[0]) + cnorm2(g[1]) + cnorm2(g[2]));
    g[0] = cscale(g[0], n0); g[1] = cscale(g[1], n0); g[2] = cscale(g[2], n0);
    // <u, m1> = sum_j conj(u_j) m_1j
    cx<T> ip = cconjmul(g[0], g[3]);
    ip = cfmaconj(g[1], g[4], ip);
    ip = cfmaconj(g[2], g[5], ip);
    g[3] = cfms(ip, g[0], g[3]);
    g[4] = cfms(ip, g[1], g[4]);
    g[5] = cfms(ip, g[2], g[5]);
    T n1 = rsqrt_t<T>(cnorm2(g[3]) + cnorm2(g[4]) + cnorm2(g[5]));
    g[3] = cscale(g[3], n1); g[4] = cscale(g[4], n1); g[5] = cscale(g[5], n1);
}

// g = reunit(m): Gram-Schmidt on rows 0, 1 of m, row 2 = conj(row0 x row1).
// m[0..5] = rows 0, 1 on entry; g[0..8] on exit.
template <typename T> __device__ __forceinline__ void reunit(cx<T> (&g)[9])
{
    reunit01<T>(g);
    su3_row2(g);
}

// Rows 0, 1 of m = 1 + a w from the 4 packed fields f0 = Im w00 + i Im w11, f1 = w01, f2 = w02,
// f3 = w12 (w anti-Hermitian traceless, so w10 = -conj(w01)); a = alpha/2 (eq. 1.2).
template <typename T>
__device__ __forceinline__ void m_from_packed(cx<T> f0, cx<T> f1, cx<T> f2, cx<T> f3, T a, cx<T> (&g)[9])
{
    g[0] = mk<T>((T)1, a * f0.x);
    g[1] = cscale(f1, a);
    g[2] = cscale(f2, a);
    g[3] = mk<T>(-a * f1.x, a * f1.y);
    g[4] = mk<T>((T)1, a * f0.y);
    g[5] = cscale(f3, a);
}

// rows [0, R) of c = a b
template <int R, typename V> __device__ __forceinline__ void mul_rows(const V (&a)[9], const V (&b)[9], V (&c)[9])
{
#pragma unroll
    for (int i = 0; i < R; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            V s = cmul(a[3 * i], b[j]);
            s = cfma(a[3 * i + 1], b[3 + j], s);
            s = cfma(a[3 * i + 2], b[6 + j], s);
            c[3 * i + j] = s;
        }
}

// rows [0, R) of c = a b^dagger
template <int R, typename V> __device__ __forceinline__ void mul_rows_dag(const V (&a)[9], const V (&b)[9], V (&c)[9])
{
#pragma unroll
    for (int i = 0; i < R; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            V s = cmulc(a[3 * i], b[3 * j]);
            s = cfmac(a[3 * i + 1], b[3 * j + 1], s);
            s = cfmac(a[3 * i + 2], b[3 * j + 2], s);
            c[3 * i + j] = s;
        }
}

// Exact exponential of eq. 1.2 as written, the variant of SURVEY 8(f4):
// rows 0, 1 of exp(A) for the anti-Hermitian traceless A = (alpha/2) w, given on entry as rows 0, 1
// of m = 1 + A (only Im m00, Im m11, m01, m02, m12 are used: the 8 real degrees of freedom).
// A traceless 3x3 matrix obeys A^3 = p A + q 1 with p = tr(A^2)/2 = -|A|_F^2/2 (real) and
// q = det A (purely imaginary), so every power is a_n 1 + b_n A + c_n A^2 with
//     a_{n+1} = q c_n,  b_{n+1} = a_n + p c_n,  c_{n+1} = b_n,
// and exp(A) = sum_n (a_n 1 + b_n A + c_n A^2)/n!.  A is first halved until |A|_F <= 1 (then 20
// terms leave a remainder below 1/21! = 2e-20) and the result squared back; no projection follows.
template <typename T> __device__ __forceinline__ void exp01_from_m(cx<T> (&g)[9])
{
    T x0 = g[0].y, x1 = g[4].y;
    cx<T> f1 = g[1], f2 = g[2], f3 = g[5];
    T n2 = x0 * x0 + x1 * x1 + (x0 + x1) * (x0 + x1) + 2 * (cnorm2(f1) + cnorm2(f2) + cnorm2(f3));
    int sq = 0;
    T sc = 1;
    while (n2 > (T)1 && sq < 60) { n2 *= (T)0.25; sc *= (T)0.5; sq++; }
    x0 *= sc; x1 *= sc; f1 = cscale(f1, sc); f2 = cscale(f2, sc); f3 = cscale(f3, sc);
    cx<T> A[9];
    A[0] = mk<T>(0, x0); A[1] = f1; A[2] = f2;
    A[3] = mk<T>(-f1.x, f1.y); A[4] = mk<T>(0, x1); A[5] = f3;
    A[6] = mk<T>(-f2.x, f2.y); A[7] = mk<T>(-f3.x, f3.y); A[8] = mk<T>(0, -(x0 + x1));
    const T p = (T)-0.5 * n2;
    // det A by the first row; its real part vanishes identically
    cx<T> c0 = cfms(A[5], A[7], cmul(A[4], A[8]));
    cx<T> c1 = cfms(A[5], A[6], cmul(A[3], A[8]));
    cx<T> c2 = cfms(A[4], A[6], cmul(A[3], A[7]));
    cx<T> det = cmul(A[0], c0);
    det = cfms(A[1], c1, det);
    det = cfma(A[2], c2, det);
    const T d = det.y;
    const double IFACT[21] = {1.0, 1.0, 0.5, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320, 1.0 / 362880,
                              1.0 / 3628800, 1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0, 1.0 / 87178291200.0,
                              1.0 / 1307674368000.0, 1.0 / 20922789888000.0, 1.0 / 355687428096000.0,
                              1.0 / 6402373705728000.0, 1.0 / 121645100408832000.0, 1.0 / 2432902008176640000.0};
    cx<T> an = mk<T>(1, 0), bn = mk<T>(0, 0), cn = mk<T>(0, 0);
    cx<T> e0 = an, e1 = bn, e2 = cn;
#pragma unroll
    for (int n = 1; n <= 20; n++) {
        const cx<T> a2 = mk<T>(-d * cn.y, d * cn.x);
        const cx<T> b2 = mk<T>(fma_t(p, cn.x, an.x), fma_t(p, cn.y, an.y));
        cn = bn; an = a2; bn = b2;
        const T f = (T)IFACT[n];
        e0.x = fma_t(f, an.x, e0.x); e0.y = fma_t(f, an.y, e0.y);
        e1.x = fma_t(f, bn.x, e1.x); e1.y = fma_t(f, bn.y, e1.y);
        e2.x = fma_t(f, cn.x, e2.x); e2.y = fma_t(f, cn.y, e2.y);
    }
    cx<T> A2[9];
    mul_rows<2>(A, A, A2);
#pragma unroll
    for (int k = 0; k < 6; k++) g[k] = cfma(e2, A2[k], cmul(e1, A[k]));
    g[0] = g[0] + e0; g[4] = g[4] + e0;
    for (int q = 0; q < sq; q++) {
        su3_row2(g);
        cx<T> t[9];
        mul_rows<2>(g, g, t);
#pragma unroll
        for (int k = 0; k < 6; k++) g[k] = t[k];
    }
}

// Rows 0, 1 of g from rows 0, 1 of m = 1 + (alpha/2) w.  gexp = 0: the paper's choice, first order
// followed by a reunitarisation; gexp = 1: the exact exponential.
template <typename T> __device__ __forceinline__ void finish_g01(cx<T> (&g)[9], int gexp)
{
    if (gexp) exp01_from_m<T>(g); else reunit01<T>(g);
}

// Rows 0, 1 of w(x) from the field buffer, then g(x) = reunit(1 + (alpha/2) w(x)), a = alpha/2
// (first order of eq. 1.2), or exp((alpha/2) w(x)) when gexp is set.
// PACK = 9: field k = 3*row+col holds w_rowcol (one FFT per matrix element, Alg. 1 line 3).
// PACK = 4: w is anti-Hermitian and traceless (the mask is real and even), so its 8 real
//   degrees of freedom are kept as  f0 = Im w00 + i Im w11,  f1 = w01,  f2 = w02,  f3 = w12;
//   then w10 = -conj(w01).
template <typename T, int PACK>
__device__ __forceinline__ void build_g(const cx<T> *__restrict__ w, int64_t V, int64_t s, T a, int gexp, cx<T> (&g)[9])
{
    if (PACK == 9) {
#pragma unroll
        for (int k = 0; k < 6; k++) g[k] = cscale(__ldg(w + (int64_t)k * V + s), a);
        g[0].x += (T)1; g[4].x += (T)1;
    } else {
        cx<T> f0 = __ldg(w + s), f1 = __ldg(w + V + s), f2 = __ldg(w + 2 * V + s), f3 = __ldg(w + 3 * V + s);
        m_from_packed<T>(f0, f1, f2, f3, a, g);
    }
    finish_g01<T>(g, gexp);
    su3_row2(g);
}

// Rows 0, 1 of g(s) (g[0..5]) for the fused kernel: read from the g buffer written by the last
// FFT pass (GBUF: 6 complex SoA arrays over sites) or built from w as above.  Row 2 is left
// to the caller (su3_row2) because not every use needs it.
template <typename T, int PACK, bool GBUF>
__device__ __forceinline__ void load_g01(const cx<T> *__restrict__ src, int64_t V, int64_t s, T a, int gexp, cx<T> (&g)[9])
{
    if (GBUF) {
#pragma unroll
        for (int k = 0; k < 6; k++) g[k] = __ldg(src + (int64_t)k * V + s);
    } else {
        if (PACK == 9) {
#pragma unroll
            for (int k = 0; k < 6; k++) g[k] = cscale(__ldg(src + (int64_t)k * V + s), a);
            g[0].x += (T)1; g[4].x += (T)1;
        } else {
            cx<T> f0 = __ldg(src + s), f1 = __ldg(src + V + s), f2 = __ldg(src + 2 * V + s), f3 = __ldg(src + 3 * V + s);
            m_from_packed<T>(f0, f1, f2, f3, a, g);
        }
        finish_g01<T>(g, gexp);
    }
}

} // namespace lgf
