// noalloc.cu -- lgf_measure_noalloc: kernel (a) of Algorithm 1 (Delta, F, theta: eq. 1.5, eq. 1.1
// PAPER.md:43, eq. 1.4) as ONE self-contained call that allocates nothing, for callers that cannot
// allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc)
// and therefore cannot set up a context with a workspace (lgf_create / lgf_bind).
//
// The measure kernel needs scratch memory: one pair of FP64 partial sums per CTA, the ticket counter of the
// fixed-order final reduction and the (F, theta) result block (reduce.cuh).  The context path carves it from the
// caller's workspace; here it lives in the file-scope device array `na_scratch` below, 131 584 bytes that every
// GPU that loads liblgf.so holds until the process exits.  That fixes the largest lattice this entry point takes:
// LGF_NOALLOC_MAX_SITES = 2^20 sites (32^4, the headline lattice) at 128 sites per CTA.
//
// In HOST code the name `na_scratch` is a host-side stand-in, not a device address: the address a kernel may use
// comes from cudaGetSymbolAddress, asked for once per device with that device current (na_scratch_ptr).
// Every call on a device shares the array and the array keeps the last call's contents: the control block is
// cleared at the start of each call (the partial sums are overwritten before they are read), and calls that
// overlap on the GPU (two streams, two host threads) race on it -- the caller must serialise them.
// No cudaMalloc, cudaFree, cudaMallocAsync or allocating library routine is called here (the only host allocation
// is the text of an error message).
#include <mutex>
#include <string>
#include "lgf.h"
#include "launch.h"
#include "su3.cuh"
#include "reduce.cuh"

namespace lgf {
namespace {

constexpr int NA_THREADS = 128;
constexpr int64_t NA_MAX_SITES = LGF_NOALLOC_MAX_SITES;
constexpr int NA_MAX_BLOCKS = (int)(NA_MAX_SITES / NA_THREADS);
// layout of the scratch array: control block | history slot of finish_measure | block partials
constexpr size_t NA_OFF_CTRL = 0, NA_OFF_HIST = 256, NA_OFF_PART = 512;
constexpr size_t NA_CLEAR_BYTES = NA_OFF_PART;                  // what must start at zero
constexpr size_t NA_SCRATCH_BYTES = NA_OFF_PART + (size_t)2 * NA_MAX_BLOCKS * sizeof(double);
static_assert(sizeof(Ctrl) <= NA_OFF_HIST && 2 * sizeof(double2) <= NA_OFF_PART - NA_OFF_HIST, "scratch layout");
static_assert(NA_SCRATCH_BYTES == LGF_NOALLOC_SCRATCH_BYTES, "include/lgf.h states the size of the scratch array");

static __device__ __align__(256) unsigned char na_scratch[NA_SCRATCH_BYTES];

// One thread per site in storage order.  links: LGF_LAYOUT_AOS [V][4][3][3]; delta (may be null): [V][3][3].
// The same arithmetic as k_measure (kernels_site.cu): A = sum_nu [U_nu(x-nu) - U_nu(x)],
// Delta = (A - A^dagger) - (1/3) Tr(A - A^dagger) (reading R3), tr F = sum_mu Re Tr U_mu(x).
template <typename T>
__global__ void __launch_bounds__(NA_THREADS)
k_measure_noalloc(const cx<T> *__restrict__ links, cx<T> *__restrict__ delta, Geom geo, unsigned char *scratch)
{
    Ctrl *ctrl = (Ctrl *)(scratch + NA_OFF_CTRL);
    double2 *hist = (double2 *)(scratch + NA_OFF_HIST);
    double *partials = (double *)(scratch + NA_OFF_PART);
    const int64_t s = (int64_t)blockIdx.x * NA_THREADS + threadIdx.x;
    double trF = 0, th = 0;
    if (s < geo.V) {
        int c[4];
        site_coords(geo, s, c);
        cx<T> A[9];
#pragma unroll
        for (int k = 0; k < 9; k++) A[k] = mk<T>(0, 0);
        T tr = 0;
#pragma unroll
        for (int nu = 0; nu < 4; nu++) {
            const int64_t sb = s + (c[nu] == 0 ? (int64_t)(geo.N[nu] - 1) : (int64_t)-1) * geo.st[nu];
            const cx<T> *pf = links + (s * 4 + nu) * 9, *pb = links + (sb * 4 + nu) * 9;
            cx<T> uf[9], ub[9];
#pragma unroll
            for (int k = 0; k < 9; k++) { uf[k] = pf[k]; ub[k] = pb[k]; }
#pragma unroll
            for (int k = 0; k < 9; k++) A[k] = A[k] + (ub[k] - uf[k]);
            tr += uf[0].x + uf[4].x + uf[8].x;
        }
        trF = (double)tr;
        T d0 = 2 * A[0].y, d1 = 2 * A[4].y, d2 = 2 * A[8].y;
        const T m = (d0 + d1 + d2) * (T)(1.0 / 3.0);
        d0 -= m; d1 -= m; d2 -= m;
        const cx<T> D01 = A[1] - cconj(A[3]), D02 = A[2] - cconj(A[6]), D12 = A[5] - cconj(A[7]);
        th = (double)(d0 * d0 + d1 * d1 + d2 * d2) + 2.0 * (double)(cnorm2(D01) + cnorm2(D02) + cnorm2(D12));
        if (delta) {
            cx<T> *o = delta + s * 9;
            o[0] = mk<T>(0, d0); o[1] = D01; o[2] = D02;
            o[3] = mk<T>(-D01.x, D01.y); o[4] = mk<T>(0, d1); o[5] = D12;
            o[6] = mk<T>(-D02.x, D02.y); o[7] = mk<T>(-D12.x, D12.y); o[8] = mk<T>(0, d2);
        }
    }
    // eps < 0: the stop flag is never raised; count_iter = 0: the result goes to hist[0]
    finish_measure<NA_THREADS>(trF, th, geo.V, ctrl, partials, hist, -1.0, 0);
}

std::mutex na_mu;
std::string na_err = "";
constexpr int NA_MAX_DEVICES = 64;
unsigned char *na_ptr[NA_MAX_DEVICES] = {};          // device address of na_scratch on each device, 0 = not asked yet

int na_fail(int code, const std::string &msg)
{
    std::lock_guard<std::mutex> lk(na_mu);
    na_err = msg;
    return code;
}

// device address of the scratch array on the CURRENT device (asked for once per device)
int na_scratch_ptr(unsigned char **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(LGF_ERR_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return na_fail(LGF_ERR_CUDA, "device index out of range");
    {
        std::lock_guard<std::mutex> lk(na_mu);
        if (na_ptr[dev]) { *out = na_ptr[dev]; return LGF_OK; }
    }
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, na_scratch);
    if (e != cudaSuccess || !p) return na_fail(LGF_ERR_CUDA, std::string("cudaGetSymbolAddress(na_scratch): ") + cudaGetErrorString(e));
    std::lock_guard<std::mutex> lk(na_mu);
    na_ptr[dev] = (unsigned char *)p;
    *out = na_ptr[dev];
    return LGF_OK;
}

} // namespace
} // namespace lgf

using namespace lgf;

extern "C" {

int lgf_measure_noalloc(int Nx, int Ny, int Nz, int Nt, int precision, const void *links_dev, void *delta_dev,
                        double *F_theta, void *cuda_stream)
{
    if (precision != LGF_PREC_FP64 && precision != LGF_PREC_FP32)
        return na_fail(LGF_ERR_INVALID_ARG, "precision must be LGF_PREC_FP64 or LGF_PREC_FP32");
    const int N[4] = {Nx, Ny, Nz, Nt};
    for (int d = 0; d < 4; d++)
        if (N[d] < 2 || N[d] > 64) return na_fail(LGF_ERR_UNSUPPORTED_SIZE, "each extent must satisfy 2 <= N <= 64");
    const int64_t V = (int64_t)Nx * Ny * Nz * Nt;
    if (V > NA_MAX_SITES)
        return na_fail(LGF_ERR_UNSUPPORTED_SIZE, "lgf_measure_noalloc: " + std::to_string(V) + " sites exceed LGF_NOALLOC_MAX_SITES = " +
                       std::to_string(NA_MAX_SITES) + " (the static scratch array holds one pair of partial sums per 128 sites); "
                       "use a context with a workspace (lgf_create, lgf_bind, lgf_measure)");
    if (!links_dev || !F_theta) return na_fail(LGF_ERR_INVALID_ARG, "links_dev and F_theta must not be NULL");
    unsigned char *scr = nullptr;
    int rc = na_scratch_ptr(&scr);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Geom g{};
    for (int d = 0; d < 4; d++) g.N[d] = N[d];
    g.st[0] = 1; g.st[1] = Nx; g.st[2] = (int64_t)Nx * Ny; g.st[3] = (int64_t)Nx * Ny * Nz;
    g.V = V; g.Vw = V; g.Vg = V; g.zb = Nz; g.Ntw = Nt; g.t0 = 0;
    // the array keeps the last call's contents: ticket, stop flag and iteration counter must start at zero
    cudaError_t e = cudaMemsetAsync(scr, 0, NA_CLEAR_BYTES, st);
    if (e != cudaSuccess) return na_fail(LGF_ERR_CUDA, std::string("cudaMemsetAsync: ") + cudaGetErrorString(e));
    const unsigned nb = (unsigned)((V + NA_THREADS - 1) / NA_THREADS);
    if (precision == LGF_PREC_FP64)
        k_measure_noalloc<double><<<nb, NA_THREADS, 0, st>>>((const cx<double> *)links_dev, (cx<double> *)delta_dev, g, scr);
    else
        k_measure_noalloc<float><<<nb, NA_THREADS, 0, st>>>((const cx<float> *)links_dev, (cx<float> *)delta_dev, g, scr);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(LGF_ERR_CUDA, std::string("k_measure_noalloc launch: ") + cudaGetErrorString(e));
    // (F, theta) are the first two doubles of the control block
    e = cudaMemcpyAsync(F_theta, scr + NA_OFF_CTRL, 2 * sizeof(double), cudaMemcpyDefault, st);
    if (e != cudaSuccess) return na_fail(LGF_ERR_CUDA, std::string("cudaMemcpyAsync(F_theta): ") + cudaGetErrorString(e));
    return LGF_OK;
}

const char *lgf_noalloc_last_error(void)
{
    std::lock_guard<std::mutex> lk(na_mu);
    static thread_local std::string copy;
    copy = na_err;
    return copy.c_str();
}

} // extern "C"
