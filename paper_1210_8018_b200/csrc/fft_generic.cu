// fft_generic.cu -- generic per-axis transform for the Fourier acceleration (Alg. 1 lines 3-8,
// PAPER.md:80-90): any even extent, one launch per axis and direction, each output of a line
// computed straight from the definition X[k] = sum_j x[j] exp(-+2 pi i j k/N) with a twiddle
// table in shared memory.  O(N^2) per line: this is the slow, size-agnostic path used for
// extents the tiled register FFT (fft_tiled.cu) does not cover, and as its cross-check.
// The mask p_max^2/p^2 (eq. 1.2; zero mode -> 0) and the 1/V normalisation are
// applied at the output of the last forward axis.
#include "launch.h"

namespace lgf {

template <typename T>
__global__ void __launch_bounds__(256)
k_fft_axis_generic(cx<T> *__restrict__ w, Geom geo, int axis, int inverse, const cx<T> *__restrict__ tw,
                   int apply_mask, const double *__restrict__ ptab, double pmax2, int LT, const Ctrl *ctrl)
{
    if (*(volatile const int *)&ctrl->done) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = geo.N[axis];
    cx<T> *tws = (cx<T> *)smem_raw;      // [N]
    cx<T> *in = tws + N;                 // [LT][N]
    const int64_t S = geo.st[axis];
    const int64_t nlines = geo.V / N;
    cx<T> *f = w + (int64_t)blockIdx.y * geo.V;
    const int tid = threadIdx.x;
    int l, j;
    if (axis == 0) { j = tid % N; l = tid / N; } else { l = tid % LT; j = tid / LT; }
    const bool active = (tid < LT * N);
    const int64_t line = (int64_t)blockIdx.x * LT + l;
    const bool ok = active && line < nlines;
    int64_t idx = 0;
    if (tid < N) {
        cx<T> t = tw[tid];
        if (inverse) t.y = -t.y;
        tws[tid] = t;
    }
    if (ok) {
        const int64_t lo = line % S, hi = line / S;
        idx = lo + hi * S * N + (int64_t)j * S;
        in[l * N + j] = f[idx];
    }
    __syncthreads();
    if (!ok) return;
    cx<T> acc = mk<T>(0, 0);
    int m = 0; // (jj * j) mod N
    for (int jj = 0; jj < N; jj++) {
        acc = cfma(in[l * N + jj], tws[m], acc);
        m += j; if (m >= N) m -= N;
    }
    if (apply_mask) {
        int c[4];
        site_coords(geo, idx, c);
        const double p2 = ptab[c[0]] + ptab[geo.N[0] + c[1]] + ptab[geo.N[0] + geo.N[1] + c[2]] +
                          ptab[geo.N[0] + geo.N[1] + geo.N[2] + c[3]];
        const T fac = (idx == 0) ? (T)0 : (T)(pmax2 / (p2 * (double)geo.V));
        acc = cscale(acc, fac);
    }
    f[idx] = acc;
}

template <typename T> static int run_generic(const FftArgs &a, cudaStream_t st)
{
    int launches = 0;
    int off[4] = {0, a.geo.N[0], a.geo.N[0] + a.geo.N[1], a.geo.N[0] + a.geo.N[1] + a.geo.N[2]};
    for (int pass = 0; pass < 8; pass++) {
        const int axis = pass < 4 ? pass : 7 - pass;
        const int inverse = pass >= 4;
        const int N = a.geo.N[axis];
        const int LT = 256 / N;
        const int64_t nlines = a.geo.V / N;
        dim3 grid((unsigned)((nlines + LT - 1) / LT), (unsigned)a.nfields);
        const size_t smem = sizeof(cx<T>) * (size_t)(N + LT * N);
        k_fft_axis_generic<T><<<grid, 256, smem, st>>>((cx<T> *)a.w, a.geo, axis, inverse, (const cx<T> *)a.tw + off[axis],
                                                       pass == 3, a.ptab, a.pmax2, LT, a.ctrl);
        launches++;
    }
    return launches;
}

int launch_fft_generic(const FftArgs &a, cudaStream_t st)
{
    return a.prec == 0 ? run_generic<double>(a, st) : run_generic<float>(a, st);
}

} // namespace lgf
