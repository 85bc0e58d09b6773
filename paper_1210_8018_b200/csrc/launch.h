// launch.h -- internal interface between the host C-ABI (lgf_api.cu) and the kernel files.
#pragma once
#include "common.cuh"

namespace lgf {

struct SiteArgs {
    Geom geo;
    void *links;        // device: cx<T> [4][NE][V]
    void *w;            // device: cx<T> [PACK][V]   (Delta, then w, in place)
    Ctrl *ctrl;         // device
    double *partials;   // device: 2 doubles per block of kernel (a)
    void *gred;         // device: group partials and group tickets of the two-level reduction (reduce.cuh, reduce2l_bytes)
    double2 *hist;      // device: LGF_HIST_CAP pairs (F, theta)
    int prec;           // 0 = FP64, 1 = FP32
    int recon;          // 18 or 12
    int pack;           // 4 or 9
    int gexp;           // LGF_OPT_GMAP: 0 first order + reunitarisation, 1 exact exponential
    int tmarch;         // LGF_OPT_TMARCH: consecutive time slices per thread of the link kernel (1, 2 or 4; divides Ntw)
    int lstream;        // LGF_OPT_LINK_STREAM resolved: 1 = the streamed link kernel (k_update_measure_stream) where the path has a g buffer
    int ltile;          // LGF_OPT_LINK_TILE resolved: 0 = one thread per site in walk order (k_update_measure), 128 / 256 / 512 = 4D tiles of that many threads
};

// kernel (a): Delta, F, theta (eq. 1.5, 1.1, 1.4).  eps < 0: never raise `done`.
void launch_measure(const SiteArgs &a, double eps, int count_iter, cudaStream_t st);
int measure_blocks(int64_t V);
// kernel (c): g(x) = reunit(1 + (alpha/2) w), U_mu(x) <- g(x) U_mu(x) g^dagger(x+mu)
void launch_update(const SiteArgs &a, double alpha, cudaStream_t st);
// kernels (c) + (a) fused: lin -> lout (distinct buffers), Delta of the new links -> wout, F, theta.
// gsrc: the g buffer (gbuf = 1: 6 complex arrays over sites) or w (gbuf = 0: a.pack fields; then wout != gsrc).
void launch_update_measure(const SiteArgs &a, const void *lin, void *lout, const void *gsrc, int gbuf, void *wout,
                           double alpha, double eps, cudaStream_t st);
int fused_blocks(int64_t V);
// threads per CTA of the tiled link kernel for this geometry, 0 when it does not apply (want = 128, 256 or 512)
int link_tile_threads(const Geom &g, int want);
// 1 when the streamed link kernel (LGF_OPT_LINK_STREAM) applies to this geometry
int link_stream_ok(const Geom &g);
// ACCUM_G (fixed links, accumulated transformation G in the g buffer, rows 0, 1):
// Delta, F, theta of G(x) U_mu(x) G^dagger(x+mu) -> a.w; counts one iteration
void launch_measure_acc(const SiteArgs &a, const void *gacc, double eps, cudaStream_t st);
// a.links <- G U G^dagger in place; then G <- 1
void launch_apply_g(const SiteArgs &a, const void *gacc, cudaStream_t st);
void launch_g_identity(const SiteArgs &a, void *gacc, cudaStream_t st);
// iter = 0, hist[0] = (F, theta), done = (theta <= eps)
void launch_ctrl_reset(const SiteArgs &a, double eps, cudaStream_t st);

// interchange layout <-> SoA, for `count` sites starting at site s0; aos points at site s0;
// per_link = 9 (LGF_LAYOUT_AOS) or 6 (LGF_LAYOUT_AOS12: rows 0, 1) complex numbers per link
void launch_aos_to_soa(const SiteArgs &a, const void *aos, int per_link, int64_t s0, int64_t count, cudaStream_t st);
void launch_soa_to_aos(const SiteArgs &a, void *aos, int per_link, int64_t s0, int64_t count, cudaStream_t st);
// site-field taps ([count][3][3] complex); which: 0 Delta / 1 w (same unpacking), 2 g
void launch_field_get(const SiteArgs &a, int which, double alpha, void *aos, int64_t s0, int64_t count, cudaStream_t st);
void launch_field_set(const SiteArgs &a, const void *aos, int64_t s0, int64_t count, cudaStream_t st);

// ---- one lattice sharded in t-slabs (LGF_OPT_SHARD_WORLD): transposes around the (z,t) pass and the global stop decision
// field buffer (4 packed fields, interior slices of the slab) <-> exchange buffer [dest rank q][t_local][field][z][y in q's range][x]
void launch_slab_pack(const SiteArgs &a, void *xbuf, int world, int unpack, cudaStream_t st);
// after the all-reduce of (F, theta): history entry of the current iteration, done = (theta <= eps) or 2 on NaN/Inf
void launch_slab_finish(const SiteArgs &a, double eps, cudaStream_t st);

// ---- Fourier acceleration (Alg. 1 lines 3-8): w <- F^-1 [p_max^2/(p^2 V)] F w, zero mode -> 0
struct FftArgs {
    Geom geo;
    void *w;            // device: cx<T> [nfields][V]
    int nfields;
    int prec;
    const double *ptab; // device: 4 sin^2(pi k/N_mu), the four tables back to back (N0+N1+N2+N3)
    double pmax2;       // max_k p^2(k)
    const void *tw;     // device: cx<T> forward twiddles exp(-2 pi i k/N_mu), four tables back to back
    const Ctrl *ctrl;
    int zt_pipe;        // LGF_OPT_ZT_PIPE: (z,t) pass as the persistent kernel with cp.async prefetch
    double vnorm;       // sites of the whole lattice: the 1/V of the inverse transform (Alg. 1 line 7)
};
// generic per-axis transform: any extent, O(N^2) per line.  Returns launches issued.
int launch_fft_generic(const FftArgs &a, cudaStream_t st);
// tiled register FFT: three passes.  which = 0 (x,y) forward, 1 (z,t) forward*mask*inverse, 2 (x,y) inverse
bool fft_tiled_supported(const int N[4], int prec);
int fft_tiled_zt_columns(const int N[4], int prec);      // x-columns per (z,t) tile, 0 if the lattice is not tiled
bool fft_tiled_gbuf_supported(const int N[4], int prec); // pass 2 with the g build fits in shared memory
void launch_fft_tiled(const FftArgs &a, int which, cudaStream_t st);
// the other pass structures of the paper's comparison (LGF_OPT_FFT_PASSES):
// 4 = 2D + 2D as four launches (step 0..3; step 3 may be replaced by launch_fft_tiled_inv_g),
// 8 = 4 x 1D as eight launches (step 0..7).  Same w as the three-pass default, to rounding.
bool fft_tiled_passes_supported(const int N[4], int prec, int passes);
void launch_fft_tiled_4pass(const FftArgs &a, int step, cudaStream_t st);
void launch_fft_tiled_8pass(const FftArgs &a, int step, cudaStream_t st);
// pass 2 of all 4 packed fields with g(x) = reunit(1 + (alpha/2) w(x)) as its epilogue: rows 0, 1 of g -> gbuf
// accum = 1: gbuf holds the accumulated G and receives reunit(g G) instead (LGF_OPT_ACCUM_G)
void launch_fft_tiled_inv_g(const FftArgs &a, void *gbuf, double alpha, int gexp, int accum, cudaStream_t st);
int fft_tiled_setup(const int N[4], int prec); // sets kernel attributes (smem opt-in); 0 on success

} // namespace lgf
