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
// Every 1D transform is done by ONE thread on a whole line held in registers: a fully
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

// ---------------------------------------------------------------- tile geometry
// Shared tile of a group: element (c, a, b) at (b*RS + a*C + c), RS = NA*C + C (one padding
// column block per row keeps 16-byte accesses of 8 consecutive threads on distinct banks).
template <int NA, int NB, int C> struct Tile {
    static constexpr int RS = NA * C + C;
    static constexpr int ELEMS = RS * NB;
    static constexpr int THREADS = C * (NA > NB ? NA : NB);
};

static const int CTA_THREADS = 128;

// ---------------------------------------------------------------- pass 0 / pass 2: (x,y) planes
// INVERSE = 0: load columns (lines along y) straight from global, Dif along y, through shared
//              memory, Dif along x, back through shared memory, coalesced store.
// INVERSE = 1: coalesced load into shared memory, Dif(+) along x, shared, Dif(+) along y,
//              store straight from registers.  Natural order in global memory in both cases.
template <typename T, int NA, int NB, int INVERSE>
__global__ void __launch_bounds__(CTA_THREADS)
k_fft_xy(cx<T> *__restrict__ w, int64_t nplanes, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    typedef Tile<NA, NB, 1> TL;
    constexpr int TP = TL::THREADS;               // threads of one plane
    constexpr int G = CTA_THREADS / TP;           // planes per CTA
    constexpr int SIGN = INVERSE ? +1 : -1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int grp = threadIdx.x / TP, t = threadIdx.x % TP;
    cx<T> *sm = (cx<T> *)smem_raw + (size_t)grp * TL::ELEMS;
    const int64_t plane = (int64_t)blockIdx.x * G + grp;
    const bool ok = plane < nplanes && grp < G;
    cx<T> *f = w + plane * (int64_t)(NA * NB);

    if (!INVERSE) {
        if (ok && t < NA) {                       // thread = x, line along y
            cx<T> v[NB];
#pragma unroll
            for (int j = 0; j < NB; j++) v[j] = f[j * NA + t];
            Dif<T, NB, NB, SIGN>::run(v);
#pragma unroll
            for (int s = 0; s < NB; s++) sm[slot_freq<NB>(s) * TL::RS + t] = v[s];
        }
        __syncthreads();
        if (ok && t < NB) {                       // thread = ky, line along x
            cx<T> v[NA];
#pragma unroll
            for (int j = 0; j < NA; j++) v[j] = sm[t * TL::RS + j];
            Dif<T, NA, NA, SIGN>::run(v);
#pragma unroll
            for (int s = 0; s < NA; s++) sm[t * TL::RS + slot_freq<NA>(s)] = v[s];
        }
        __syncthreads();
        if (ok && t < NA) {
#pragma unroll
            for (int j = 0; j < NB; j++) f[j * NA + t] = sm[j * TL::RS + t];
        }
    } else {
        if (ok && t < NA) {
#pragma unroll
            for (int j = 0; j < NB; j++) sm[j * TL::RS + t] = f[j * NA + t];
        }
        __syncthreads();
        if (ok && t < NB) {
            cx<T> v[NA];
#pragma unroll
            for (int j = 0; j < NA; j++) v[j] = sm[t * TL::RS + j];
            Dif<T, NA, NA, SIGN>::run(v);
#pragma unroll
            for (int s = 0; s < NA; s++) sm[t * TL::RS + slot_freq<NA>(s)] = v[s];
        }
        __syncthreads();
        if (ok && t < NA) {
            cx<T> v[NB];
#pragma unroll
            for (int j = 0; j < NB; j++) v[j] = sm[j * TL::RS + t];
            Dif<T, NB, NB, SIGN>::run(v);
#pragma unroll
            for (int s = 0; s < NB; s++) f[slot_freq<NB>(s) * NA + t] = v[s];
        }
    }
}

// ---------------------------------------------------------------- pass 2 with the g build fused
// (x,y) inverse of all four packed fields of one (z,t) plane in one CTA, then
// g(x) = reunit(1 + (alpha/2) w(x)) (Alg. 1 lines 9-11) straight from shared
// memory: w never goes back to HBM, rows 0, 1 of g (12 reals) do.  The fused link kernel
// (kernels_fused.cu) then reads g at x and its 8 neighbours instead of rebuilding it 9 times.
template <typename T, int NA, int NB>
__global__ void __launch_bounds__(CTA_THREADS)
k_fft_xy_inv_g(const cx<T> *__restrict__ w, cx<T> *__restrict__ gbuf, int64_t V, int64_t nplanes, T a, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    typedef Tile<NA, NB, 1> TL;
    constexpr int TP = TL::THREADS;               // threads of one field of one plane
    constexpr int TG = 4 * TP;                    // threads of one plane
    constexpr int G = CTA_THREADS / TG;           // planes per CTA
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int grp = threadIdx.x / TG, t = threadIdx.x % TG;
    const int fld = t / TP, l = t % TP;
    cx<T> *smp = (cx<T> *)smem_raw + (size_t)grp * 4 * TL::ELEMS;   // the 4 fields of this plane
    cx<T> *sm = smp + (size_t)fld * TL::ELEMS;
    const int64_t plane = (int64_t)blockIdx.x * G + grp;
    const bool ok = plane < nplanes && grp < G;
    const int64_t base = plane * (int64_t)(NA * NB);

    if (ok && l < NA) {
        const cx<T> *f = w + (int64_t)fld * V + base;
#pragma unroll
        for (int j = 0; j < NB; j++) sm[j * TL::RS + l] = f[j * NA + l];
    }
    __syncthreads();
    if (ok && l < NB) {
        cx<T> v[NA];
#pragma unroll
        for (int j = 0; j < NA; j++) v[j] = sm[l * TL::RS + j];
        Dif<T, NA, NA, +1>::run(v);
#pragma unroll
        for (int s = 0; s < NA; s++) sm[l * TL::RS + slot_freq<NA>(s)] = v[s];
    }
    __syncthreads();
    if (ok && l < NA) {
        cx<T> v[NB];
#pragma unroll
        for (int j = 0; j < NB; j++) v[j] = sm[j * TL::RS + l];
        Dif<T, NB, NB, +1>::run(v);
#pragma unroll
        for (int s = 0; s < NB; s++) sm[slot_freq<NB>(s) * TL::RS + l] = v[s];
    }
    __syncthreads();
    if (ok) {
        for (int i = t; i < NA * NB; i += TG) {
            const int o = (i / NA) * TL::RS + (i % NA);
            cx<T> g[9];
            m_from_packed<T>(smp[o], smp[TL::ELEMS + o], smp[2 * TL::ELEMS + o], smp[3 * TL::ELEMS + o], a, g);
            reunit01<T>(g);
            cx<T> *dst = gbuf + base + i;
#pragma unroll
            for (int k = 0; k < 6; k++) dst[(int64_t)k * V] = g[k];
        }
    }
}

// ---------------------------------------------------------------- pass 1: (z,t) tiles
// Tile = C consecutive x at fixed (field, y): element (c, z, t) at global x0 + c + sz*z + st*t.
// z-lines straight from global (thread = (c, t)), Dif(-) along z -> shared; t-lines from
// shared (thread = (c, kz)): Dif(-), mask, Dit(+) -> shared; z-lines from shared: Dif(+),
// stored straight to global.  p^2 = sum_mu 4 sin^2(pi k_mu/N_mu) (reading R5) from the
// per-axis tables; the factor p_max^2/(p^2 V) is one FP64 division per mode.
template <typename T, int NA, int NB, int C>
__global__ void __launch_bounds__(CTA_THREADS)
k_fft_zt(cx<T> *__restrict__ w, Geom geo, const double *__restrict__ ptab, double pmax2_over_V, int64_t ntiles, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    typedef Tile<NA, NB, C> TL;
    constexpr int TT = TL::THREADS;
    constexpr int G = CTA_THREADS / TT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *pt = (double *)smem_raw;                                  // 4 sin^2(pi kt/Nt), NB entries
    cx<T> *sm0 = (cx<T> *)(smem_raw + ((NB * sizeof(double) + 15) / 16) * 16);
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
    if (threadIdx.x < NB) pt[threadIdx.x] = ptab[Nx + Ny + NA + threadIdx.x];
    const int c = t % C, l = t / C;                                    // l = t-index or z-index of the line

    if (ok && l < NB) {                                                // z-lines, thread = (c, t = l)
        cx<T> v[NA];
        const cx<T> *g = f + c + st * l;
#pragma unroll
        for (int j = 0; j < NA; j++) v[j] = g[sz * j];
        Dif<T, NA, NA, -1>::run(v);
#pragma unroll
        for (int s = 0; s < NA; s++) sm[l * TL::RS + slot_freq<NA>(s) * C + c] = v[s];
    }
    __syncthreads();
    if (ok && l < NA) {                                                // t-lines, thread = (c, kz = l)
        cx<T> v[NB];
#pragma unroll
        for (int j = 0; j < NB; j++) v[j] = sm[j * TL::RS + l * C + c];
        Dif<T, NB, NB, -1>::run(v);
        const double pxyz = ptab[x0 + c] + ptab[Nx + y] + ptab[Nx + Ny + l];
#pragma unroll
        for (int s = 0; s < NB; s++) {
            const double p2 = pxyz + pt[slot_freq<NB>(s)];
            const T fac = (p2 > 0.0) ? (T)(pmax2_over_V / p2) : (T)0;  // zero mode -> 0 (reading R7)
            v[s] = cscale(v[s], fac);
        }
        Dit<T, NB, NB, +1>::run(v);
#pragma unroll
        for (int j = 0; j < NB; j++) sm[j * TL::RS + l * C + c] = v[j];
    }
    __syncthreads();
    if (ok && l < NB) {
        cx<T> v[NA];
#pragma unroll
        for (int j = 0; j < NA; j++) v[j] = sm[l * TL::RS + j * C + c];
        Dif<T, NA, NA, +1>::run(v);
        cx<T> *g = f + c + st * l;
#pragma unroll
        for (int s = 0; s < NA; s++) g[sz * slot_freq<NA>(s)] = v[s];
    }
}

// ---------------------------------------------------------------- dispatch
template <typename T, int NA, int NB> struct XYCfg {
    typedef Tile<NA, NB, 1> TL;
    static constexpr int G = CTA_THREADS / TL::THREADS;
    static constexpr size_t SMEM = (size_t)G * TL::ELEMS * sizeof(cx<T>);
};
template <typename T, int NA, int NB> struct XYGCfg {
    typedef Tile<NA, NB, 1> TL;
    static constexpr int G = CTA_THREADS / (4 * TL::THREADS);
    static constexpr size_t SMEM = (size_t)G * 4 * TL::ELEMS * sizeof(cx<T>);
};
template <typename T, int NA, int NB, int C> struct ZTCfg {
    typedef Tile<NA, NB, C> TL;
    static constexpr int G = CTA_THREADS / TL::THREADS;
    static constexpr size_t SMEM = ((NB * sizeof(double) + 15) / 16) * 16 + (size_t)G * TL::ELEMS * sizeof(cx<T>);
};

static const int ZT_C = 4; // x-columns per (z,t) tile: 64-byte (FP64) runs in global memory

template <typename T, int N> static int setup_n()
{
    cudaError_t e;
    e = cudaFuncSetAttribute(k_fft_xy<T, N, N, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYCfg<T, N, N>::SMEM);
    if (e != cudaSuccess) return 1;
    e = cudaFuncSetAttribute(k_fft_xy<T, N, N, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYCfg<T, N, N>::SMEM);
    if (e != cudaSuccess) return 1;
    e = cudaFuncSetAttribute(k_fft_xy_inv_g<T, N, N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XYGCfg<T, N, N>::SMEM);
    if (e != cudaSuccess) return 1;
    e = cudaFuncSetAttribute(k_fft_zt<T, N, N, ZT_C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZTCfg<T, N, N, ZT_C>::SMEM);
    if (e != cudaSuccess) return 1;
    return 0;
}

template <typename T, int N> static void launch_n(const FftArgs &a, int which, cudaStream_t st)
{
    if (which == 1) {
        typedef ZTCfg<T, N, N, ZT_C> Z;
        const int64_t ntiles = (int64_t)a.nfields * a.geo.N[1] * (a.geo.N[0] / ZT_C);
        const unsigned grid = (unsigned)((ntiles + Z::G - 1) / Z::G);
        k_fft_zt<T, N, N, ZT_C><<<grid, CTA_THREADS, Z::SMEM, st>>>((cx<T> *)a.w, a.geo, a.ptab, a.pmax2 / (double)a.geo.V, ntiles, a.ctrl);
    } else {
        typedef XYCfg<T, N, N> X;
        const int64_t nplanes = (int64_t)a.nfields * a.geo.N[2] * a.geo.N[3];
        const unsigned grid = (unsigned)((nplanes + X::G - 1) / X::G);
        if (which == 0) k_fft_xy<T, N, N, 0><<<grid, CTA_THREADS, X::SMEM, st>>>((cx<T> *)a.w, nplanes, a.ctrl);
        else k_fft_xy<T, N, N, 1><<<grid, CTA_THREADS, X::SMEM, st>>>((cx<T> *)a.w, nplanes, a.ctrl);
    }
}

template <typename T, int N> static void launch_inv_g_n(const FftArgs &a, void *gbuf, double alpha, cudaStream_t st)
{
    typedef XYGCfg<T, N, N> X;
    const int64_t nplanes = (int64_t)a.geo.N[2] * a.geo.N[3];
    const unsigned grid = (unsigned)((nplanes + X::G - 1) / X::G);
    k_fft_xy_inv_g<T, N, N><<<grid, CTA_THREADS, X::SMEM, st>>>((const cx<T> *)a.w, (cx<T> *)gbuf, a.geo.V, nplanes, (T)(alpha / 2.0), a.ctrl);
}

// Hypercubic N^4 lattices whose lines fit in registers: N = 8, 16, 32 in both precisions,
// N = 12, 24 (radix 3 x 2^a).  Everything else takes the generic path.
bool fft_tiled_supported(const int N[4], int prec)
{
    (void)prec;
    if (!(N[0] == N[1] && N[1] == N[2] && N[2] == N[3])) return false;
    return N[0] == 8 || N[0] == 16 || N[0] == 32 || N[0] == 12 || N[0] == 24;
}

#define LGF_FFT_SWITCH(FN, ...)                                         \
    switch (n) {                                                        \
    case 8: return prec == 0 ? FN<double, 8>(__VA_ARGS__) : FN<float, 8>(__VA_ARGS__);    \
    case 12: return prec == 0 ? FN<double, 12>(__VA_ARGS__) : FN<float, 12>(__VA_ARGS__); \
    case 16: return prec == 0 ? FN<double, 16>(__VA_ARGS__) : FN<float, 16>(__VA_ARGS__); \
    case 24: return prec == 0 ? FN<double, 24>(__VA_ARGS__) : FN<float, 24>(__VA_ARGS__); \
    case 32: return prec == 0 ? FN<double, 32>(__VA_ARGS__) : FN<float, 32>(__VA_ARGS__); \
    default: break;                                                     \
    }

int fft_tiled_setup(const int N[4], int prec)
{
    const int n = N[0];
    LGF_FFT_SWITCH(setup_n)
    return 1;
}

void launch_fft_tiled(const FftArgs &a, int which, cudaStream_t st)
{
    const int n = a.geo.N[0], prec = a.prec;
    LGF_FFT_SWITCH(launch_n, a, which, st)
}

// pass 2 fused with the g build: needs the 4 packed fields (nfields == 4)
void launch_fft_tiled_inv_g(const FftArgs &a, void *gbuf, double alpha, cudaStream_t st)
{
    const int n = a.geo.N[0], prec = a.prec;
    LGF_FFT_SWITCH(launch_inv_g_n, a, gbuf, alpha, st)
}

} // namespace lgf
