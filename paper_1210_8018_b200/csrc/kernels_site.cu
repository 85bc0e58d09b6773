// kernels_site.cu -- the per-site kernels of one gauge-fixing iteration (arXiv 1210.8018):
//   kernel (a) k_measure : Delta(x) (eq. 1.5), F (eq. 1.1), theta (eq. 1.4)
//   kernel (c) k_update  : g(x) = reunit(1 + (alpha/2) w(x)) and
//                          U_mu(x) <- g(x) U_mu(x) g^dagger(x+mu)  (Alg. 1 lines 9-16)
// plus the layout conversions and debug taps of the C ABI.  One thread per lattice site;
// links and fields are complex SoA arrays over sites, so every load of a warp is one
// contiguous run of 16-byte (FP64) or 8-byte (FP32) complex numbers.
#include "launch.h"
#include "su3.cuh"
#include "reduce.cuh"

namespace lgf {

static const int SITE_THREADS = 128;

// ------------------------------------------------------------------ kernel (a)
// A = sum_nu [U_nu(x-nu) - U_nu(x)];  Delta = (A - A^dagger) - (1/3) Tr(A - A^dagger) 1  (reading R3).
// Per-site Re Tr sum_mu U_mu(x) and Tr Delta Delta^dagger are reduced in FP64: warp shuffles,
// one partial per block, and the last block to finish adds the partials in index order.
// The last block also takes the stop decision of Alg. 1 line 2 (theta <= eps).
template <typename T, int NE, int PACK>
__global__ void __launch_bounds__(SITE_THREADS)
k_measure(const cx<T> *__restrict__ links, cx<T> *__restrict__ w, Geom geo, Ctrl *ctrl,
          double *partials, double2 *hist, double eps, int count_iter)
{
    if (*(volatile int *)&ctrl->done) return;
    const int64_t V = geo.V;
    const int64_t rr = (int64_t)blockIdx.x * SITE_THREADS + threadIdx.x;
    double trF = 0, th = 0;
    if (rr < geo.Vw) {
        int c[4];
        const int64_t s = walk_site(geo, rr, c);
        cx<T> A[9];
#pragma unroll
        for (int k = 0; k < 9; k++) A[k] = mk<T>(0, 0);
        T tr = 0;
#pragma unroll
        for (int nu = 0; nu < 4; nu++) {
            const int64_t sb = s + (c[nu] == 0 ? (int64_t)(geo.N[nu] - 1) : (int64_t)-1) * geo.st[nu];
            cx<T> uf[9], ub[9];
            load_link<T, NE>(links, V, nu, s, uf);
            load_link<T, NE>(links, V, nu, sb, ub);
#pragma unroll
            for (int k = 0; k < 9; k++) A[k] = A[k] + (ub[k] - uf[k]);
            tr += uf[0].x + uf[4].x + uf[8].x;
        }
        trF = (double)tr;
        // D = A - A^dagger: D_ii = 2i Im A_ii, D_ij = A_ij - conj(A_ji); remove the trace
        T d0 = 2 * A[0].y, d1 = 2 * A[4].y, d2 = 2 * A[8].y;
        const T m = (d0 + d1 + d2) * (T)(1.0 / 3.0);
        d0 -= m; d1 -= m; d2 -= m;
        cx<T> D01 = A[1] - cconj(A[3]), D02 = A[2] - cconj(A[6]), D12 = A[5] - cconj(A[7]);
        th = (double)(d0 * d0 + d1 * d1 + d2 * d2) + 2.0 * (double)(cnorm2(D01) + cnorm2(D02) + cnorm2(D12));
        if (PACK == 4) {
            w[s] = mk<T>(d0, d1);
            w[V + s] = D01;
            w[2 * V + s] = D02;
            w[3 * V + s] = D12;
        } else {
            w[s] = mk<T>(0, d0);
            w[V + s] = D01;
            w[2 * V + s] = D02;
            w[3 * V + s] = mk<T>(-D01.x, D01.y);
            w[4 * V + s] = mk<T>(0, d1);
            w[5 * V + s] = D12;
            w[6 * V + s] = mk<T>(-D02.x, D02.y);
            w[7 * V + s] = mk<T>(-D12.x, D12.y);
            w[8 * V + s] = mk<T>(0, d2);
        }
    }
    finish_measure<SITE_THREADS>(trF, th, geo.Vg, ctrl, partials, hist, eps, count_iter);
}

__global__ void k_ctrl_reset(Ctrl *ctrl, double2 *hist, double eps)
{
    ctrl->iter = 0;
    hist[0] = make_double2(ctrl->F, ctrl->theta);
    const double theta = ctrl->theta;
    ctrl->done = (!(theta == theta) || theta > 1.0e300) ? 2 : (theta <= eps ? 1 : 0);
}

// ------------------------------------------------------------------ kernel (c)
// Every g comes from the w of the previous measure (Jacobi update, reading R14); g(x+mu) is
// rebuilt from w(x+mu) instead of being stored, so each link is read once and written once.
// With 12-real storage only rows 0, 1 of g U g^dagger are computed and stored (reading R15).
template <typename T, int NE, int PACK>
__global__ void __launch_bounds__(SITE_THREADS)
k_update(cx<T> *links, const cx<T> *__restrict__ w, Geom geo, T a, int gexp, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    const int64_t V = geo.V;
    const int64_t rr = (int64_t)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (rr >= geo.Vw) return;
    int c[4];
    const int64_t s = walk_site(geo, rr, c);
    cx<T> g0[9];
    build_g<T, PACK>(w, V, s, a, gexp, g0);
    constexpr int R = (NE == 6) ? 2 : 3;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const int64_t sp = s + (c[mu] == geo.N[mu] - 1 ? -(int64_t)(geo.N[mu] - 1) : (int64_t)1) * geo.st[mu];
        cx<T> g1[9], u[9], t[9], r[9];
        build_g<T, PACK>(w, V, sp, a, gexp, g1);
        load_link_rw<T, NE>(links, V, mu, s, u);
        mul_rows<R>(g0, u, t);
        mul_rows_dag<R>(t, g1, r);
        cx<T> *p = links + (int64_t)mu * NE * V + s;
#pragma unroll
        for (int k = 0; k < NE; k++) p[(int64_t)k * V] = r[k];
    }
}

// ------------------------------------------------------------------ ACCUM_G: apply the accumulated G
// U_mu(x) <- G(x) U_mu(x) G^dagger(x+mu) in place, from the rows 0, 1 of G kept in the g buffer
// (LGF_OPT_ACCUM_G; the same product as k_update, Alg. 1 lines 12-16, with the
// accumulated transformation in place of one iteration's g).  Each thread rewrites only its own
// four links and G is read-only here; k_g_identity resets it afterwards.
template <typename T, int NE>
__global__ void __launch_bounds__(SITE_THREADS)
k_apply_g(cx<T> *links, const cx<T> *__restrict__ gacc, Geom geo)
{
    const int64_t V = geo.V;
    const int64_t rr = (int64_t)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (rr >= geo.Vw) return;
    int c[4];
    const int64_t s = walk_site(geo, rr, c);
    cx<T> g0[9];
    load_g01<T, 4, true>(gacc, V, s, (T)0, 0, g0);
    su3_row2(g0);
    constexpr int R = (NE == 6) ? 2 : 3;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const int64_t sp = s + (c[mu] == geo.N[mu] - 1 ? -(int64_t)(geo.N[mu] - 1) : (int64_t)1) * geo.st[mu];
        cx<T> g1[9], u[9], t[9], r[9];
        load_g01<T, 4, true>(gacc, V, sp, (T)0, 0, g1);
        su3_row2(g1);
        load_link_rw<T, NE>(links, V, mu, s, u);
        mul_rows<R>(g0, u, t);
        mul_rows_dag<R>(t, g1, r);
        cx<T> *p = links + (int64_t)mu * NE * V + s;
#pragma unroll
        for (int k = 0; k < NE; k++) p[(int64_t)k * V] = r[k];
    }
}

template <typename T> __global__ void k_g_identity(cx<T> *__restrict__ gacc, int64_t V)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= V) return;
#pragma unroll
    for (int k = 0; k < 6; k++) gacc[(int64_t)k * V + s] = mk<T>((k == 0 || k == 4) ? (T)1 : (T)0, (T)0);
}

// ------------------------------------------------------------------ one lattice sharded in t-slabs
// Transposes around the (z,t) pass (the all-to-all of a distributed FFT, as PFFT does for the paper's CPU
// program).  A rank holds Ntl time slices of every field; for the (z,t) pass it needs
// ALL time slices of the sites with y in its range of Ny/world rows.  Pack: the interior slices of the 4 packed
// fields -> the send buffer, ordered [destination q][t_local][field][z][y - q Nyl][x], so that the block for q
// is contiguous; after the all-to-all the receive buffer reads [source r][t_local][field][z][y_local][x] =
// [t][field][z][y_local][x], which is the array the (z,t) kernel runs on (field stride Nx Nyl Nz, t stride 4 times
// that).  Unpack is the same map backwards after the return all-to-all.  Consecutive threads: consecutive x.
template <typename T, int UNPACK>
__global__ void k_slab_pack(cx<T> *__restrict__ w, cx<T> *__restrict__ xbuf, Geom geo, int world)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= 4 * geo.Vw) return;
    const int Nx = geo.N[0], Ny = geo.N[1], Nz = geo.N[2], Ntl = geo.Ntw, Nyl = Ny / world;
    unsigned u = (unsigned)e;
    const int x = (int)(u % (unsigned)Nx); u /= (unsigned)Nx;
    const int y = (int)(u % (unsigned)Ny); u /= (unsigned)Ny;
    const int z = (int)(u % (unsigned)Nz); u /= (unsigned)Nz;
    const int tl = (int)(u % (unsigned)Ntl); u /= (unsigned)Ntl;
    const int f = (int)u;
    const int q = y / Nyl, yl = y % Nyl;
    const int64_t iw = (int64_t)f * geo.V + x + (int64_t)Nx * y + geo.st[2] * z + geo.st[3] * (tl + geo.t0);
    const int64_t ix = ((((int64_t)q * Ntl + tl) * 4 + f) * Nz + z) * ((int64_t)Nyl * Nx) + (int64_t)yl * Nx + x;
    if (UNPACK) w[iw] = xbuf[ix]; else xbuf[ix] = w[iw];
}

// (F, theta) in the control block are the sums over all ranks now: history entry of the current iteration
// and the stop decision of Alg. 1 line 2, the same on every rank.
__global__ void k_slab_finish(Ctrl *ctrl, double2 *hist, double eps)
{
    const double F = ctrl->F, theta = ctrl->theta;
    const long long it = ctrl->iter;
    if (it < LGF_HIST_CAP) hist[it] = make_double2(F, theta);
    if (!(theta == theta) || theta > 1.0e300) ctrl->done = 2;
    else if (theta <= eps) ctrl->done = 1;
}

// ------------------------------------------------------------------ layout conversions and taps
// PER = complex numbers per link in the interchange array: 9 (LGF_LAYOUT_AOS) or 6 (LGF_LAYOUT_AOS12,
// rows 0, 1; row 2 = conj(row0 x row1) is rebuilt here when the links are stored with 18 reals).
template <typename T, int NE, int PER>
__global__ void k_aos_to_soa(const cx<T> *__restrict__ aos, cx<T> *__restrict__ links, int64_t V, int64_t s0, int64_t count)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count * 4) return;
    const int mu = (int)(i / count);
    const int64_t sl = i % count;
    const cx<T> *src = aos + (sl * 4 + mu) * PER;
    cx<T> *dst = links + (int64_t)mu * NE * V + s0 + sl;
    cx<T> u[9];
#pragma unroll
    for (int k = 0; k < (NE < PER ? NE : PER); k++) u[k] = src[k];
    if (NE > PER) su3_row2(u);
#pragma unroll
    for (int k = 0; k < NE; k++) dst[(int64_t)k * V] = u[k];
}

template <typename T, int NE, int PER>
__global__ void k_soa_to_aos(cx<T> *__restrict__ aos, const cx<T> *__restrict__ links, int64_t V, int64_t s0, int64_t count)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count * 4) return;
    const int mu = (int)(i / count);
    const int64_t sl = i % count;
    cx<T> u[9];
    load_link<T, NE>(links, V, mu, s0 + sl, u);
    cx<T> *dst = aos + (sl * 4 + mu) * PER;
#pragma unroll
    for (int k = 0; k < PER; k++) dst[k] = u[k];
}

template <typename T, int PACK>
__global__ void k_field_get(const cx<T> *__restrict__ w, int64_t V, int which, T a, int gexp, cx<T> *__restrict__ aos, int64_t s0, int64_t count)
{
    const int64_t sl = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (sl >= count) return;
    const int64_t s = s0 + sl;
    cx<T> m[9];
    if (which == 2) {
        build_g<T, PACK>(w, V, s, a, gexp, m);
    } else if (PACK == 9) {
#pragma unroll
        for (int k = 0; k < 9; k++) m[k] = w[(int64_t)k * V + s];
    } else {
        cx<T> f0 = w[s], f1 = w[V + s], f2 = w[2 * V + s], f3 = w[3 * V + s];
        m[0] = mk<T>(0, f0.x); m[4] = mk<T>(0, f0.y); m[8] = mk<T>(0, -(f0.x + f0.y));
        m[1] = f1; m[2] = f2; m[5] = f3;
        m[3] = mk<T>(-f1.x, f1.y); m[6] = mk<T>(-f2.x, f2.y); m[7] = mk<T>(-f3.x, f3.y);
    }
#pragma unroll
    for (int k = 0; k < 9; k++) aos[sl * 9 + k] = m[k];
}

template <typename T, int PACK>
__global__ void k_field_set(cx<T> *__restrict__ w, int64_t V, const cx<T> *__restrict__ aos, int64_t s0, int64_t count)
{
    const int64_t sl = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (sl >= count) return;
    const int64_t s = s0 + sl;
    const cx<T> *m = aos + sl * 9;
    if (PACK == 9) {
#pragma unroll
        for (int k = 0; k < 9; k++) w[(int64_t)k * V + s] = m[k];
    } else {
        w[s] = mk<T>(m[0].y, m[4].y);
        w[V + s] = m[1];
        w[2 * V + s] = m[2];
        w[3 * V + s] = m[5];
    }
}

// ------------------------------------------------------------------ dispatch
int measure_blocks(int64_t V) { return (int)((V + SITE_THREADS - 1) / SITE_THREADS); }

#define LGF_DISPATCH(CALL)                                                              \
    do {                                                                                \
        if (a.prec == 0) {                                                              \
            if (a.recon == 12) { if (a.pack == 4) { CALL(double, 6, 4); } else { CALL(double, 6, 9); } } \
            else               { if (a.pack == 4) { CALL(double, 9, 4); } else { CALL(double, 9, 9); } } \
        } else {                                                                        \
            if (a.recon == 12) { if (a.pack == 4) { CALL(float, 6, 4); } else { CALL(float, 6, 9); } }   \
            else               { if (a.pack == 4) { CALL(float, 9, 4); } else { CALL(float, 9, 9); } }   \
        }                                                                               \
    } while (0)

void launch_measure(const SiteArgs &a, double eps, int count_iter, cudaStream_t st)
{
    const int nb = measure_blocks(a.geo.Vw);
#define CALL(T, NE, PACK) \
    k_measure<T, NE, PACK><<<nb, SITE_THREADS, 0, st>>>((const cx<T> *)a.links, (cx<T> *)a.w, a.geo, a.ctrl, a.partials, a.hist, eps, count_iter)
    LGF_DISPATCH(CALL);
#undef CALL
}

void launch_update(const SiteArgs &a, double alpha, cudaStream_t st)
{
    const int nb = measure_blocks(a.geo.Vw);
#define CALL(T, NE, PACK) \
    k_update<T, NE, PACK><<<nb, SITE_THREADS, 0, st>>>((cx<T> *)a.links, (const cx<T> *)a.w, a.geo, (T)(alpha / 2.0), a.gexp, a.ctrl)
    LGF_DISPATCH(CALL);
#undef CALL
}

void launch_apply_g(const SiteArgs &a, const void *gacc, cudaStream_t st)
{
    const int nb = measure_blocks(a.geo.Vw);
#define CALL(T, NE, PACK) \
    k_apply_g<T, NE><<<nb, SITE_THREADS, 0, st>>>((cx<T> *)a.links, (const cx<T> *)gacc, a.geo)
    LGF_DISPATCH(CALL);
#undef CALL
}

void launch_g_identity(const SiteArgs &a, void *gacc, cudaStream_t st)
{
    const int nb = (int)((a.geo.V + 255) / 256);
    if (a.prec == 0) k_g_identity<double><<<nb, 256, 0, st>>>((cx<double> *)gacc, a.geo.V);
    else k_g_identity<float><<<nb, 256, 0, st>>>((cx<float> *)gacc, a.geo.V);
}

void launch_slab_pack(const SiteArgs &a, void *xbuf, int world, int unpack, cudaStream_t st)
{
    const int nb = (int)((4 * a.geo.Vw + 255) / 256);
    if (a.prec == 0) {
        if (unpack) k_slab_pack<double, 1><<<nb, 256, 0, st>>>((cx<double> *)a.w, (cx<double> *)xbuf, a.geo, world);
        else k_slab_pack<double, 0><<<nb, 256, 0, st>>>((cx<double> *)a.w, (cx<double> *)xbuf, a.geo, world);
    } else {
        if (unpack) k_slab_pack<float, 1><<<nb, 256, 0, st>>>((cx<float> *)a.w, (cx<float> *)xbuf, a.geo, world);
        else k_slab_pack<float, 0><<<nb, 256, 0, st>>>((cx<float> *)a.w, (cx<float> *)xbuf, a.geo, world);
    }
}

void launch_slab_finish(const SiteArgs &a, double eps, cudaStream_t st)
{
    k_slab_finish<<<1, 1, 0, st>>>(a.ctrl, a.hist, eps);
}

void launch_ctrl_reset(const SiteArgs &a, double eps, cudaStream_t st)
{
    k_ctrl_reset<<<1, 1, 0, st>>>(a.ctrl, a.hist, eps);
}

void launch_aos_to_soa(const SiteArgs &a, const void *aos, int per_link, int64_t s0, int64_t count, cudaStream_t st)
{
    s0 += a.geo.t0 * a.geo.st[3];     // sharded lattice: the interchange arrays hold the interior slices only
    const int nb = (int)((count * 4 + 255) / 256);
#define CALL(T, NE, PACK) \
    do { if (per_link == 6) k_aos_to_soa<T, NE, 6><<<nb, 256, 0, st>>>((const cx<T> *)aos, (cx<T> *)a.links, a.geo.V, s0, count); \
         else k_aos_to_soa<T, NE, 9><<<nb, 256, 0, st>>>((const cx<T> *)aos, (cx<T> *)a.links, a.geo.V, s0, count); } while (0)
    LGF_DISPATCH(CALL);
#undef CALL
}

void launch_soa_to_aos(const SiteArgs &a, void *aos, int per_link, int64_t s0, int64_t count, cudaStream_t st)
{
    s0 += a.geo.t0 * a.geo.st[3];     // sharded lattice: the interchange arrays hold the interior slices only
    const int nb = (int)((count * 4 + 255) / 256);
#define CALL(T, NE, PACK) \
    do { if (per_link == 6) k_soa_to_aos<T, NE, 6><<<nb, 256, 0, st>>>((cx<T> *)aos, (const cx<T> *)a.links, a.geo.V, s0, count); \
         else k_soa_to_aos<T, NE, 9><<<nb, 256, 0, st>>>((cx<T> *)aos, (const cx<T> *)a.links, a.geo.V, s0, count); } while (0)
    LGF_DISPATCH(CALL);
#undef CALL
}

void launch_field_get(const SiteArgs &a, int which, double alpha, void *aos, int64_t s0, int64_t count, cudaStream_t st)
{
    s0 += a.geo.t0 * a.geo.st[3];
    const int nb = (int)((count + 255) / 256);
#define CALL(T, NE, PACK) \
    k_field_get<T, PACK><<<nb, 256, 0, st>>>((const cx<T> *)a.w, a.geo.V, which, (T)(alpha / 2.0), a.gexp, (cx<T> *)aos, s0, count)
    LGF_DISPATCH(CALL);
#undef CALL
}

void launch_field_set(const SiteArgs &a, const void *aos, int64_t s0, int64_t count, cudaStream_t st)
{
    s0 += a.geo.t0 * a.geo.st[3];
    const int nb = (int)((count + 255) / 256);
#define CALL(T, NE, PACK) \
    k_field_set<T, PACK><<<nb, 256, 0, st>>>((cx<T> *)a.w, a.geo.V, (const cx<T> *)aos, s0, count)
    LGF_DISPATCH(CALL);
#undef CALL
}

} // namespace lgf
