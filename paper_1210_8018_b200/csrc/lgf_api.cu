// lgf_api.cu -- host side of liblgf.so: the C ABI declared in include/lgf.h.
// Owns no device memory: carves the caller's workspace, launches the kernels of
// kernels_site.cu / fft_tiled.cu / fft_generic.cu on the caller's stream, and keeps the
// loop of Algorithm 1 on the device between polls of the `done` flag.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/lgf.h"
#include "launch.h"
#include "reduce.cuh"

using namespace lgf;

static_assert(LGF_HIST_CAP == LGF_HISTORY_CAP, "history capacity: common.cuh and lgf.h must agree");

namespace {

const double kTwoPi = 6.283185307179586476925286766559;
std::string g_create_err = "";

struct EvPair { cudaEvent_t a, b; int kind; };

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Layout {
    size_t links[2], w[2], gbuf, partials, gred, ctrl, hist, ptab, tw, staging, xbuf[2], ptab_zt, total;
    int64_t staging_sites;
};

} // namespace

struct lgf_ctx {
    int N[4];
    int64_t V;
    int prec;
    int recon = 18, pack = 4, check_interval = 8, fft_path = 0, profile = 0, fusion = 1, l2_persist = 0, gmap = 0, accum = 0;
    int graph = 1;           // LGF_OPT_GRAPH: replay captured iterations as a CUDA graph
    int zblock = 0;          // LGF_OPT_ZBLOCK: 0 = auto (resolved by lgf_bind into sa.geo.zb)
    int zt_pipe = 0;         // LGF_OPT_ZT_PIPE
    int fft_passes = 3;      // LGF_OPT_FFT_PASSES: 3 (fused middle), 4 (2D + 2D), 8 (4 x 1D)
    int tmarch = 0;          // LGF_OPT_TMARCH: time slices per thread of the link kernel (0 = auto)
    int link_tile = 0;       // LGF_OPT_LINK_TILE: 0 / 1 = off, 128 / 256 / 512 threads per tile
    int link_stream = 0;     // LGF_OPT_LINK_STREAM: 1 = TMA-fed persistent link kernel
    // one lattice sharded in t-slabs over shard_world ranks (0 = off): V = sites of the interchange arrays (the
    // rank's own time slices), Vp = stored sites (with the two halo slices), Vg = sites of the whole lattice
    int shard_world = 0, shard_rank = 0;
    int64_t Vp = 0, Vg = 0;
    void *xbuf[2] = {nullptr, nullptr};   // exchange buffers of the transposes (send, receive)
    FftArgs fa_zt{};                      // the (z,t) pass on the transposed field
    cudaGraphExec_t gexec = nullptr;
    struct { double alpha, eps; int cur, wcur, gmap, unit; } gkey{};
    int64_t g_launches = 0, g_kcount[LGF_KERNEL_KINDS] = {0};
    bool acc_dirty = false;  // ACCUM_G: the g buffer holds a G != 1 that the links do not yet include
    bool l2_window = false;  // an access-policy window is set on the bound stream
    int cur = 0, wcur = 0;   // which of the two link / field buffers is current
    bool use_gbuf = false;   // last FFT pass writes g (fusion, tiled FFT, 4 packed fields)
    void *links_buf[2] = {nullptr, nullptr}, *w_buf[2] = {nullptr, nullptr}, *gbuf = nullptr;
    int64_t max_iter = 100000;
    bool bound = false, loaded = false;
    int wstate = 0; // 0 invalid, 1 holds Delta of the current links, 2 holds w
    cudaStream_t st = nullptr;
    char *base = nullptr;
    Layout lay{};
    SiteArgs sa{};
    FftArgs fa{};
    bool tiled = false;
    std::vector<double> ptab_h;
    double pmax2 = 0;
    int64_t launches = 0;
    std::vector<EvPair> evs;
    size_t ev_used = 0;
    double kms[LGF_KERNEL_KINDS] = {0};
    int64_t kcount[LGF_KERNEL_KINDS] = {0};
    std::string err;
};

namespace {

size_t elem_bytes(const lgf_ctx *c) { return c->prec == LGF_PREC_FP64 ? 16 : 8; }
int sum_n(const lgf_ctx *c) { return c->N[0] + c->N[1] + c->N[2] + c->N[3]; }

Layout make_layout(const lgf_ctx *c)
{
    Layout L{};
    const size_t e = elem_bytes(c);
    const int ne = c->recon == 12 ? 6 : 9;
    size_t off = 0;
    // sharded: the arrays hold the rank's Nt / world time slices plus one halo slice on either side
    const int64_t plane3 = (int64_t)c->N[0] * c->N[1] * c->N[2];
    const int64_t Vl = c->shard_world > 0 ? plane3 * (c->N[3] / c->shard_world) : (int64_t)plane3 * c->N[3];
    const int64_t Vs = c->shard_world > 0 ? Vl + 2 * plane3 : Vl;
    // fusion: links are double-buffered (the fused kernel reads old neighbours while new links
    // are written); the fields are double-buffered when g is rebuilt from w inside that kernel,
    // else the last FFT pass writes rows 0, 1 of g (6 complex per site) to gbuf
    // ACCUM_G: the links are not rewritten per iteration, so one buffer; the g buffer holds G
    const int nl = (c->fusion && !c->accum) ? 2 : 1;
    const bool gb = c->fusion && c->pack == 4 && c->fft_path == 0 && c->fft_passes != 8 && fft_tiled_gbuf_supported(c->N, c->prec);
    const int nw = (c->fusion && !gb) ? 2 : 1;
    for (int i = 0; i < 2; i++) { L.links[i] = off; if (i < nl) off = align_up(off + (size_t)4 * ne * Vs * e, 256); }
    for (int i = 0; i < 2; i++) { L.w[i] = off; if (i < nw) off = align_up(off + (size_t)c->pack * Vs * e, 256); }
    L.gbuf = off; if (gb) off = align_up(off + (size_t)6 * Vs * e, 256);
    // the tiled link kernel (LGF_OPT_LINK_TILE) may leave threads of a CTA idle: at most twice the CTAs (link_tile_threads checks)
    const int nblk = std::max(measure_blocks(Vl), 2 * fused_blocks(Vl) + 2);
    L.partials = off; off = align_up(off + (size_t)2 * nblk * sizeof(double), 256);
    L.gred = off; off = align_up(off + reduce2l_bytes(fused_blocks(Vl)), 256);
    L.ctrl = off; off = align_up(off + sizeof(Ctrl), 256);
    L.hist = off; off = align_up(off + (size_t)LGF_HIST_CAP * sizeof(double2), 256);
    L.ptab = off; off = align_up(off + (size_t)sum_n(c) * sizeof(double), 256);
    L.tw = off; off = align_up(off + (size_t)sum_n(c) * e, 256);
    L.staging_sites = Vl < (1 << 17) ? Vl : (1 << 17);
    L.staging = off; off = align_up(off + (size_t)L.staging_sites * 36 * e, 256);
    for (int i = 0; i < 2; i++) { L.xbuf[i] = off; if (c->shard_world > 0) off = align_up(off + (size_t)4 * Vl * e, 256); }
    L.ptab_zt = off; if (c->shard_world > 0) off = align_up(off + (size_t)sum_n(c) * sizeof(double), 256);
    L.total = off;
    return L;
}

int fail(lgf_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg; else g_create_err = msg;
    return code;
}

int cuda_fail(lgf_ctx *c, cudaError_t e, const char *what)
{
    return fail(c, LGF_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define CK(call)                                                   \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);   \
    } while (0)

bool smooth23(int n)
{
    while (n % 2 == 0) n /= 2;
    while (n % 3 == 0) n /= 3;
    return n == 1;
}

// bracket a launch with events when profiling
template <typename F> void run_kernel(lgf_ctx *c, int kind, int nlaunch, F f)
{
    if (c->profile) {
        if (c->ev_used == c->evs.size()) {
            EvPair p;
            cudaEventCreate(&p.a);
            cudaEventCreate(&p.b);
            p.kind = kind;
            c->evs.push_back(p);
        }
        EvPair &p = c->evs[c->ev_used++];
        p.kind = kind;
        cudaEventRecord(p.a, c->st);
        f();
        cudaEventRecord(p.b, c->st);
    } else {
        f();
    }
    c->launches += nlaunch;
    c->kcount[kind] += nlaunch;
}

void flush_events(lgf_ctx *c)
{
    if (!c->ev_used) return;
    cudaStreamSynchronize(c->st);
    for (size_t i = 0; i < c->ev_used; i++) {
        float ms = 0;
        if (cudaEventElapsedTime(&ms, c->evs[i].a, c->evs[i].b) == cudaSuccess) c->kms[c->evs[i].kind] += ms;
    }
    c->ev_used = 0;
}

void sync_ptrs(lgf_ctx *c)
{
    c->sa.links = c->links_buf[c->cur];
    c->sa.w = c->w_buf[c->wcur];
    c->fa.w = c->sa.w;
}

void do_measure(lgf_ctx *c, double eps, int count_iter)
{
    run_kernel(c, LGF_KERNEL_MEASURE, 1, [&] { launch_measure(c->sa, eps, count_iter, c->st); });
    c->wstate = 1;
}

// the tiled FFT up to, but without, its last (x,y) inverse pass, in the pass structure LGF_OPT_FFT_PASSES asks for
void do_fourier_head(lgf_ctx *c)
{
    if (c->fft_passes == 4) {
        run_kernel(c, LGF_KERNEL_FFT_XY_FWD, 1, [&] { launch_fft_tiled_4pass(c->fa, 0, c->st); });
        run_kernel(c, LGF_KERNEL_FFT_ZT, 2, [&] { launch_fft_tiled_4pass(c->fa, 1, c->st); launch_fft_tiled_4pass(c->fa, 2, c->st); });
    } else {
        run_kernel(c, LGF_KERNEL_FFT_XY_FWD, 1, [&] { launch_fft_tiled(c->fa, 0, c->st); });
        run_kernel(c, LGF_KERNEL_FFT_ZT, 1, [&] { launch_fft_tiled(c->fa, 1, c->st); });
    }
}

void do_fourier(lgf_ctx *c)
{
    if (c->tiled && c->fft_passes == 8) {
        run_kernel(c, LGF_KERNEL_FFT_XY_FWD, 2, [&] { launch_fft_tiled_8pass(c->fa, 0, c->st); launch_fft_tiled_8pass(c->fa, 1, c->st); });
        run_kernel(c, LGF_KERNEL_FFT_ZT, 4, [&] { for (int s = 2; s < 6; s++) launch_fft_tiled_8pass(c->fa, s, c->st); });
        run_kernel(c, LGF_KERNEL_FFT_XY_INV, 2, [&] { launch_fft_tiled_8pass(c->fa, 6, c->st); launch_fft_tiled_8pass(c->fa, 7, c->st); });
    } else if (c->tiled) {
        do_fourier_head(c);
        run_kernel(c, LGF_KERNEL_FFT_XY_INV, 1, [&] { launch_fft_tiled(c->fa, 2, c->st); });
    } else {
        run_kernel(c, LGF_KERNEL_FFT_GENERIC, 8, [&] { launch_fft_generic(c->fa, c->st); });
    }
    c->wstate = 2;
}

void do_update(lgf_ctx *c, double alpha)
{
    run_kernel(c, LGF_KERNEL_UPDATE, 1, [&] { launch_update(c->sa, alpha, c->st); });
    c->wstate = 0;
}

// ACCUM_G: bring the links up to date, U <- G U G^dagger, G <- 1.  The field buffer keeps the Delta of
// these links (wstate unchanged).  No-op when nothing is pending.
void materialise(lgf_ctx *c)
{
    if (!c->accum || !c->acc_dirty) return;
    run_kernel(c, LGF_KERNEL_APPLY_G, 2, [&] {
        launch_apply_g(c->sa, c->gbuf, c->st);
        launch_g_identity(c->sa, c->gbuf, c->st);
    });
    c->acc_dirty = false;
}

// one execution of the loop body of Algorithm 1 (lines 3-17) on the device
void do_iteration(lgf_ctx *c, double alpha, double eps)
{
    if (c->accum) {
        // w_buf[0] holds Delta of G U G^dagger; the last FFT pass turns it into g and G <- g G
        do_fourier_head(c);
        run_kernel(c, LGF_KERNEL_FFT_XY_INV_GACC, 1, [&] { launch_fft_tiled_inv_g(c->fa, c->gbuf, alpha, c->gmap, 1, c->st); });
        run_kernel(c, LGF_KERNEL_MEASURE_ACC, 1, [&] { launch_measure_acc(c->sa, c->gbuf, eps, c->st); });
        c->acc_dirty = true;
        c->wstate = 1;
        return;
    }
    if (!c->fusion) {
        do_fourier(c);
        do_update(c, alpha);
        do_measure(c, eps, 1);
        return;
    }
    // w_buf[wcur] holds Delta of links_buf[cur]
    void *lin = c->links_buf[c->cur], *lout = c->links_buf[c->cur ^ 1];
    if (c->use_gbuf) {
        do_fourier_head(c);
        run_kernel(c, LGF_KERNEL_FFT_XY_INV_G, 1, [&] { launch_fft_tiled_inv_g(c->fa, c->gbuf, alpha, c->gmap, 0, c->st); });
        run_kernel(c, LGF_KERNEL_UPDATE_MEASURE, 1,
                   [&] { launch_update_measure(c->sa, lin, lout, c->gbuf, 1, c->w_buf[c->wcur], alpha, eps, c->st); });
    } else {
        do_fourier(c);
        void *win = c->w_buf[c->wcur], *wout = c->w_buf[c->wcur ^ 1];
        run_kernel(c, LGF_KERNEL_UPDATE_MEASURE, 1,
                   [&] { launch_update_measure(c->sa, lin, lout, win, 0, wout, alpha, eps, c->st); });
        c->wcur ^= 1;
    }
    c->cur ^= 1;
    sync_ptrs(c);
    c->wstate = 1;
}

void graph_drop(lgf_ctx *c)
{
    if (c->gexec) cudaGraphExecDestroy(c->gexec);
    c->gexec = nullptr;
}

bool graph_matches(const lgf_ctx *c, double alpha, double eps, int unit)
{
    return c->gexec && c->gkey.alpha == alpha && c->gkey.eps == eps && c->gkey.cur == c->cur && c->gkey.wcur == c->wcur &&
           c->gkey.gmap == c->gmap && c->gkey.unit == unit;
}

// Capture `unit` iterations (even: the double buffers are back where they started) into a graph.
// Kernel arguments (alpha, eps, buffer pointers, g map) are baked in, so they key the cached graph.
// Nothing is enqueued.  Any failure switches the graph path off for this context; the direct
// launches remain.
void graph_capture(lgf_ctx *c, double alpha, double eps, int unit)
{
    graph_drop(c);
    const int cur0 = c->cur, wcur0 = c->wcur, ws0 = c->wstate;
    const bool dirty0 = c->acc_dirty;
    const int64_t l0 = c->launches;
    int64_t k0[LGF_KERNEL_KINDS];
    for (int k = 0; k < LGF_KERNEL_KINDS; k++) k0[k] = c->kcount[k];
    if (cudaStreamBeginCapture(c->st, cudaStreamCaptureModeRelaxed) != cudaSuccess) { cudaGetLastError(); c->graph = 0; return; }
    for (int i = 0; i < unit; i++) do_iteration(c, alpha, eps);
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->st, &g);
    c->g_launches = c->launches - l0;
    c->launches = l0;
    for (int k = 0; k < LGF_KERNEL_KINDS; k++) { c->g_kcount[k] = c->kcount[k] - k0[k]; c->kcount[k] = k0[k]; }
    const bool back = (c->cur == cur0 && c->wcur == wcur0);
    c->cur = cur0; c->wcur = wcur0; c->wstate = ws0; c->acc_dirty = dirty0;
    sync_ptrs(c);
    if (e == cudaSuccess && g && back) e = cudaGraphInstantiate(&c->gexec, g, 0);
    if (g) cudaGraphDestroy(g);
    if (e != cudaSuccess || !c->gexec || !back) { cudaGetLastError(); graph_drop(c); c->graph = 0; return; }
    c->gkey.alpha = alpha; c->gkey.eps = eps; c->gkey.cur = cur0; c->gkey.wcur = wcur0; c->gkey.gmap = c->gmap; c->gkey.unit = unit;
}

// n executions of the loop body.  With a cached graph of the same arguments: whole units as graph
// replays, the rest as direct launches.  Without one: direct launches now, and the graph for the
// next call (or the next poll interval of lgf_fix) is captured afterwards, while the GPU is busy with
// these launches, so that capture and instantiation never sit in front of the work.
void run_iterations(lgf_ctx *c, double alpha, double eps, int64_t n)
{
    const int unit = 2 * std::max(1, std::min(c->check_interval, 8) / 2);
    const bool want = c->graph && !c->profile && n >= unit;
    if (want && graph_matches(c, alpha, eps, unit)) {
        while (n >= unit) {
            if (cudaGraphLaunch(c->gexec, c->st) != cudaSuccess) { cudaGetLastError(); graph_drop(c); c->graph = 0; break; }
            c->launches += c->g_launches;
            for (int k = 0; k < LGF_KERNEL_KINDS; k++) c->kcount[k] += c->g_kcount[k];
            c->wstate = 1;
            if (c->accum) c->acc_dirty = true;
            n -= unit;
        }
        for (int64_t i = 0; i < n; i++) do_iteration(c, alpha, eps);
        return;
    }
    for (int64_t i = 0; i < n; i++) do_iteration(c, alpha, eps);
    if (want && c->graph) graph_capture(c, alpha, eps, unit);
}

// Kernels launched after the device raised `done` exit without writing, so after a poll the
// current buffers are those of the `executed`-th iteration since `cur0` / `wcur0`.
void settle_buffers(lgf_ctx *c, int cur0, int wcur0, long long executed)
{
    if (!c->fusion || c->accum) return;
    c->cur = cur0 ^ (int)(executed & 1);
    if (!c->use_gbuf) c->wcur = wcur0 ^ (int)(executed & 1);
    sync_ptrs(c);
}

int read_ctrl(lgf_ctx *ctx, Ctrl *h)
{
    CK(cudaMemcpyAsync(h, ctx->sa.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, ctx->st));
    CK(cudaStreamSynchronize(ctx->st));
    CK(cudaGetLastError());
    return LGF_OK;
}

int clear_done(lgf_ctx *ctx)
{
    CK(cudaMemsetAsync(&ctx->sa.ctrl->done, 0, sizeof(int), ctx->st));
    return LGF_OK;
}

// L2 residency of the field buffer: Delta is written by the link kernel, then read and written by
// the three FFT passes; it is far smaller than the links (64 of 1344 bytes per site), so keeping it
// in the persisting part of L2 removes its HBM round trips.  Best effort: silently skipped when
// the device has no persisting L2 or the buffer does not fit.
void l2_window_set(lgf_ctx *c)
{
    c->l2_window = false;
    if (!c->l2_persist) return;
    int dev = 0, max_persist = 0, max_window = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return;
    cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, dev);
    cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, dev);
    const size_t bytes = (size_t)c->pack * c->V * elem_bytes(c);
    if (max_persist <= 0 || bytes > (size_t)max_persist || bytes > (size_t)max_window) { cudaGetLastError(); return; }
    if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, bytes) != cudaSuccess) { cudaGetLastError(); return; }
    cudaStreamAttrValue v{};
    v.accessPolicyWindow.base_ptr = c->w_buf[0];
    v.accessPolicyWindow.num_bytes = bytes;
    v.accessPolicyWindow.hitRatio = 1.0f;
    v.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    v.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    if (cudaStreamSetAttribute(c->st, cudaStreamAttributeAccessPolicyWindow, &v) != cudaSuccess) { cudaGetLastError(); return; }
    c->l2_window = true;
}

void l2_window_clear(lgf_ctx *c)
{
    if (!c->l2_window) return;
    cudaStreamAttrValue v{};
    v.accessPolicyWindow.num_bytes = 0;
    cudaStreamSetAttribute(c->st, cudaStreamAttributeAccessPolicyWindow, &v);
    cudaCtxResetPersistingL2Cache();
    cudaGetLastError();
    c->l2_window = false;
}

// LGF_OPT_ZBLOCK = 0: the largest divisor of Nz such that one z-block of (x,y) planes, with everything the
// link kernel streams per site (links in and out, g, Delta), takes at most LGF_ZBLOCK_L2_FRACTION of L2.
// The reuse distance of a -t / +t neighbour is one z-block of planes, so it has to stay well inside L2
// together with the write-back lines of the new links.  Falls back to Nz (storage order) when the L2 size
// cannot be read.
#ifndef LGF_ZBLOCK_L2_FRACTION
#define LGF_ZBLOCK_L2_FRACTION 0.38
#endif
int auto_zblock(const lgf_ctx *c)
{
    int dev = 0, l2 = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev) != cudaSuccess || l2 <= 0) {
        cudaGetLastError();
        return c->N[2];
    }
    const size_t e = elem_bytes(c);
    const int ne = c->recon == 12 ? 6 : 9;
    const size_t per_site = (size_t)(2 * 4 * ne + 6 + c->pack) * e;
    const double plane = (double)c->N[0] * c->N[1] * (double)per_site;
    int best = 1;
    for (int zb = 1; zb <= c->N[2]; zb++)
        if (c->N[2] % zb == 0 && zb * plane <= LGF_ZBLOCK_L2_FRACTION * (double)l2) best = zb;
    return best;
}

int need_loaded(lgf_ctx *ctx)
{
    if (!ctx) return LGF_ERR_INVALID_ARG;
    if (!ctx->bound) return fail(ctx, LGF_ERR_NOT_BOUND, "lgf_bind has not been called");
    if (!ctx->loaded) return fail(ctx, LGF_ERR_NOT_LOADED, "lgf_load_links has not been called");
    return LGF_OK;
}

// the single-GPU drivers (measure / iterate / fix / stage / field taps) see only this rank's slab
int need_unsharded(lgf_ctx *ctx)
{
    int rc = need_loaded(ctx);
    if (rc) return rc;
    if (ctx->shard_world > 0) return fail(ctx, LGF_ERR_INVALID_ARG, "sharded context (SHARD_WORLD): drive it with lgf_shard_step");
    return LGF_OK;
}

} // namespace

extern "C" {

int lgf_create(int Nx, int Ny, int Nz, int Nt, int precision, lgf_ctx **out)
{
    if (!out) return fail(nullptr, LGF_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (precision != LGF_PREC_FP64 && precision != LGF_PREC_FP32)
        return fail(nullptr, LGF_ERR_INVALID_ARG, "precision must be LGF_PREC_FP64 or LGF_PREC_FP32");
    const int N[4] = {Nx, Ny, Nz, Nt};
    for (int d = 0; d < 4; d++)
        if (N[d] < 4 || N[d] > 64 || (N[d] & 1) || !smooth23(N[d]))
            return fail(nullptr, LGF_ERR_UNSUPPORTED_SIZE, "each extent must be even, 4 <= N <= 64, of the form 2^a 3^b");
    lgf_ctx *c = new (std::nothrow) lgf_ctx;
    if (!c) return fail(nullptr, LGF_ERR_INVALID_ARG, "out of host memory");
    for (int d = 0; d < 4; d++) c->N[d] = N[d];
    c->V = (int64_t)Nx * Ny * Nz * Nt;
    c->prec = precision;
    // s_mu[k] = 4 sin^2(pi k/N_mu): eigenvalues of minus the lattice second difference
    // (reading R5); p_max^2 = sum_mu max_k s_mu[k] (reading R6).
    c->pmax2 = 0;
    for (int d = 0; d < 4; d++) {
        double m = 0;
        for (int k = 0; k < N[d]; k++) {
            const double sn = std::sin(0.5 * kTwoPi * (double)k / (double)N[d]);
            const double v = 4.0 * sn * sn;
            c->ptab_h.push_back(v);
            if (v > m) m = v;
        }
        c->pmax2 += m;
    }
    *out = c;
    return LGF_OK;
}

int lgf_set_option(lgf_ctx *ctx, int key, int64_t value)
{
    if (!ctx) return LGF_ERR_INVALID_ARG;
    const bool layout_key = (key == LGF_OPT_RECON || key == LGF_OPT_FFT_BATCH || key == LGF_OPT_FFT_PATH || key == LGF_OPT_FUSION ||
                             key == LGF_OPT_L2_PERSIST || key == LGF_OPT_ACCUM_G || key == LGF_OPT_ZBLOCK || key == LGF_OPT_FFT_PASSES ||
                             key == LGF_OPT_SHARD_WORLD || key == LGF_OPT_SHARD_RANK || key == LGF_OPT_TMARCH || key == LGF_OPT_LINK_TILE || key == LGF_OPT_LINK_STREAM);
    if (layout_key && ctx->bound) return fail(ctx, LGF_ERR_INVALID_ARG, "this option must be set before lgf_bind");
    switch (key) {
    case LGF_OPT_RECON:
        if (value != 12 && value != 18) return fail(ctx, LGF_ERR_INVALID_ARG, "RECON must be 12 or 18");
        ctx->recon = (int)value; break;
    case LGF_OPT_FFT_BATCH:
        if (value != 4 && value != 9) return fail(ctx, LGF_ERR_INVALID_ARG, "FFT_BATCH must be 4 or 9");
        ctx->pack = (int)value; break;
    case LGF_OPT_MAX_ITER:
        if (value < 0) return fail(ctx, LGF_ERR_INVALID_ARG, "MAX_ITER must be >= 0");
        ctx->max_iter = value; break;
    case LGF_OPT_CHECK_INTERVAL:
        if (value < 1 || value > 1024) return fail(ctx, LGF_ERR_INVALID_ARG, "CHECK_INTERVAL must be in 1..1024");
        ctx->check_interval = (int)value; break;
    case LGF_OPT_FFT_PATH:
        if (value != 0 && value != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "FFT_PATH must be 0 or 1");
        ctx->fft_path = (int)value; break;
    case LGF_OPT_FUSION:
        if (value != 0 && value != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "FUSION must be 0 or 1");
        ctx->fusion = (int)value; break;
    case LGF_OPT_L2_PERSIST:
        if (value != 0 && value != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "L2_PERSIST must be 0 or 1");
        ctx->l2_persist = (int)value; break;
    case LGF_OPT_GMAP:
        if (value != 0 && value != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "GMAP must be 0 or 1");
        ctx->gmap = (int)value; ctx->sa.gexp = ctx->gmap; break;
    case LGF_OPT_ACCUM_G:
        if (value != 0 && value != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "ACCUM_G must be 0 or 1");
        ctx->accum = (int)value; break;
    case LGF_OPT_GRAPH:
        if (value != 0 && value != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "GRAPH must be 0 or 1");
        ctx->graph = (int)value; break;
    case LGF_OPT_ZBLOCK:
        if (value < 0 || (value > 0 && ctx->N[2] % value != 0)) return fail(ctx, LGF_ERR_INVALID_ARG, "ZBLOCK must be 0 (auto) or a divisor of Nz");
        ctx->zblock = (int)value; break;
    case LGF_OPT_FFT_PASSES:
        if (value != 3 && value != 4 && value != 8) return fail(ctx, LGF_ERR_INVALID_ARG, "FFT_PASSES must be 3, 4 or 8");
        ctx->fft_passes = (int)value; break;
    case LGF_OPT_TMARCH:
        if (value != 0 && value != 1 && value != 2 && value != 4) return fail(ctx, LGF_ERR_INVALID_ARG, "TMARCH must be 0 (auto), 1, 2 or 4");
        ctx->tmarch = (int)value; break;
    case LGF_OPT_LINK_TILE:
        if (value != 0 && value != 1 && value != 128 && value != 256 && value != 512)
            return fail(ctx, LGF_ERR_INVALID_ARG, "LINK_TILE must be 0 or 1 (off), 128, 256 or 512");
        ctx->link_tile = (int)value; break;
    case LGF_OPT_LINK_STREAM:
        if (value != 0 && value != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "LINK_STREAM must be 0 or 1");
        ctx->link_stream = (int)value; break;
    case LGF_OPT_SHARD_WORLD:
        if (value < 0 || (value > 0 && (ctx->N[3] % value != 0 || ctx->N[1] % value != 0)))
            return fail(ctx, LGF_ERR_INVALID_ARG, "SHARD_WORLD must be 0 (off) or divide Nt and Ny");
        ctx->shard_world = (int)value; if (ctx->shard_rank >= value) ctx->shard_rank = 0; break;
    case LGF_OPT_SHARD_RANK:
        if (value < 0 || value >= std::max(1, ctx->shard_world)) return fail(ctx, LGF_ERR_INVALID_ARG, "SHARD_RANK must be in [0, SHARD_WORLD)");
        ctx->shard_rank = (int)value; break;
    case LGF_OPT_ZT_PIPE:
        if (value != 0 && value != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "ZT_PIPE must be 0 or 1");
        ctx->zt_pipe = (int)value; ctx->fa.zt_pipe = ctx->zt_pipe; graph_drop(ctx); break;
    case LGF_OPT_PROFILE:
        if (ctx->bound) flush_events(ctx);
        ctx->profile = value ? 1 : 0; break;
    default:
        return fail(ctx, LGF_ERR_INVALID_ARG, "unknown option key");
    }
    return LGF_OK;
}

size_t lgf_workspace_bytes(const lgf_ctx *ctx)
{
    if (!ctx) return 0;
    return make_layout(ctx).total;
}

int lgf_bind(lgf_ctx *ctx, void *dev_workspace, size_t bytes, void *cuda_stream)
{
    if (!ctx) return LGF_ERR_INVALID_ARG;
    if (!dev_workspace) return fail(ctx, LGF_ERR_INVALID_ARG, "dev_workspace is NULL");
    if (((uintptr_t)dev_workspace) & 255) return fail(ctx, LGF_ERR_INVALID_ARG, "dev_workspace must be 256-byte aligned");
    if (ctx->accum && !(ctx->fusion && ctx->pack == 4 && ctx->fft_path == 0 && fft_tiled_gbuf_supported(ctx->N, ctx->prec)))
        return fail(ctx, LGF_ERR_INVALID_ARG, "ACCUM_G needs FUSION = 1, FFT_BATCH = 4 and a lattice the tiled FFT covers");
    if (ctx->fft_passes != 3 && !(ctx->fft_path == 0 && fft_tiled_passes_supported(ctx->N, ctx->prec, ctx->fft_passes)))
        return fail(ctx, LGF_ERR_INVALID_ARG, "FFT_PASSES = 4 / 8 need a lattice the tiled FFT covers (4: a square or 32 x n (z,t) tile)");
    if (ctx->fft_passes == 8 && ctx->accum)
        return fail(ctx, LGF_ERR_INVALID_ARG, "ACCUM_G builds g in the last 2D pass: not available with FFT_PASSES = 8");
    if (ctx->shard_world > 0 && !(ctx->fusion && ctx->pack == 4 && ctx->fft_path == 0 && ctx->fft_passes == 3 && !ctx->accum &&
                                  fft_tiled_gbuf_supported(ctx->N, ctx->prec)))
        return fail(ctx, LGF_ERR_INVALID_ARG, "SHARD_WORLD needs the default path: FUSION = 1, FFT_BATCH = 4, FFT_PASSES = 3, no ACCUM_G, a lattice the tiled FFT covers");
    const Layout L = make_layout(ctx);
    if (bytes < L.total) return fail(ctx, LGF_ERR_WORKSPACE_TOO_SMALL, "workspace smaller than lgf_workspace_bytes()");
    ctx->lay = L;
    ctx->base = (char *)dev_workspace;
    ctx->st = (cudaStream_t)cuda_stream;
    Geom g{};
    for (int d = 0; d < 4; d++) g.N[d] = ctx->N[d];
    g.st[0] = 1; g.st[1] = g.N[0]; g.st[2] = (int64_t)g.N[0] * g.N[1]; g.st[3] = (int64_t)g.N[0] * g.N[1] * g.N[2];
    g.zb = ctx->zblock > 0 ? ctx->zblock : auto_zblock(ctx);
    ctx->Vg = g.st[3] * ctx->N[3];
    if (ctx->shard_world > 0) {
        const int ntl = ctx->N[3] / ctx->shard_world;
        ctx->V = g.st[3] * ntl;                 // the interchange arrays of this rank: its own time slices
        ctx->Vp = g.st[3] * (ntl + 2);
        g.N[3] = ntl + 2; g.Ntw = ntl; g.t0 = 1;
    } else {
        ctx->V = ctx->Vg; ctx->Vp = ctx->Vg;
        g.Ntw = g.N[3]; g.t0 = 0;
    }
    g.V = ctx->Vp; g.Vw = ctx->V; g.Vg = ctx->Vg;
    SiteArgs &s = ctx->sa;
    s.geo = g;
    // auto: measured on B200 (profiles/r02_link_kernel.md) FP32 gains 3 % with 4 slices per thread, FP64 loses 15 % (the
    // carried product costs registers the FP64 kernel does not have: 364 B of spills); the walked slices must split into whole groups
    const int want = ctx->tmarch > 0 ? ctx->tmarch : ((ctx->prec == LGF_PREC_FP32 && !ctx->accum) ? 4 : 1);
    s.tmarch = (g.Ntw % want == 0) ? want : 1;
    s.ltile = (ctx->link_tile > 1 && ctx->fusion && !ctx->accum) ? link_tile_threads(g, ctx->link_tile) : 0;
    s.lstream = (ctx->link_stream == 1 && ctx->fusion && !ctx->accum) ? link_stream_ok(g) : 0;
    for (int i = 0; i < 2; i++) { ctx->links_buf[i] = ctx->base + L.links[i]; ctx->w_buf[i] = ctx->base + L.w[i]; }
    ctx->gbuf = ctx->base + L.gbuf;
    ctx->cur = 0; ctx->wcur = 0;
    s.partials = (double *)(ctx->base + L.partials);
    s.gred = ctx->base + L.gred;
    s.ctrl = (Ctrl *)(ctx->base + L.ctrl);
    s.hist = (double2 *)(ctx->base + L.hist);
    s.prec = ctx->prec; s.recon = ctx->recon; s.pack = ctx->pack; s.gexp = ctx->gmap;
    FftArgs &f = ctx->fa;
    f.geo = g; f.nfields = ctx->pack; f.prec = ctx->prec; f.zt_pipe = ctx->zt_pipe; f.vnorm = (double)ctx->Vg;
    sync_ptrs(ctx);
    f.ptab = (const double *)(ctx->base + L.ptab);
    f.pmax2 = ctx->pmax2;
    f.tw = ctx->base + L.tw;
    f.ctrl = s.ctrl;
    // tables: momentum tables and forward twiddles exp(-2 pi i k/N), computed in FP64, rounded once (R19)
    const int sn = sum_n(ctx);
    CK(cudaMemcpyAsync(ctx->base + L.ptab, ctx->ptab_h.data(), sizeof(double) * sn, cudaMemcpyHostToDevice, ctx->st));
    std::vector<double> twd(2 * sn);
    std::vector<float> twf(2 * sn);
    int o = 0;
    for (int d = 0; d < 4; d++)
        for (int k = 0; k < ctx->N[d]; k++, o++) {
            const double ang = kTwoPi * (double)k / (double)ctx->N[d];
            twd[2 * o] = std::cos(ang); twd[2 * o + 1] = -std::sin(ang);
            twf[2 * o] = (float)twd[2 * o]; twf[2 * o + 1] = (float)twd[2 * o + 1];
        }
    if (ctx->prec == LGF_PREC_FP64) CK(cudaMemcpyAsync(ctx->base + L.tw, twd.data(), sizeof(double) * 2 * sn, cudaMemcpyHostToDevice, ctx->st));
    else CK(cudaMemcpyAsync(ctx->base + L.tw, twf.data(), sizeof(float) * 2 * sn, cudaMemcpyHostToDevice, ctx->st));
    if (ctx->shard_world > 0) {
        // the (z,t) pass runs on the transposed field: all Nt time slices of the sites with y in this rank's range
        const int R = ctx->shard_world, nyl = ctx->N[1] / R;
        for (int i = 0; i < 2; i++) ctx->xbuf[i] = ctx->base + L.xbuf[i];
        FftArgs &z = ctx->fa_zt;
        z = f;
        z.geo.N[1] = nyl; z.geo.N[3] = ctx->N[3];
        z.geo.V = (int64_t)ctx->N[0] * nyl * ctx->N[2];                   // field stride
        z.geo.st[1] = ctx->N[0]; z.geo.st[2] = (int64_t)ctx->N[0] * nyl; z.geo.st[3] = 4 * z.geo.V;
        z.w = ctx->xbuf[1];
        std::vector<double> pz;                                            // the y table restricted to this rank's rows
        pz.insert(pz.end(), ctx->ptab_h.begin(), ctx->ptab_h.begin() + ctx->N[0]);
        pz.insert(pz.end(), ctx->ptab_h.begin() + ctx->N[0] + ctx->shard_rank * nyl, ctx->ptab_h.begin() + ctx->N[0] + (ctx->shard_rank + 1) * nyl);
        pz.insert(pz.end(), ctx->ptab_h.begin() + ctx->N[0] + ctx->N[1], ctx->ptab_h.end());
        CK(cudaMemcpyAsync(ctx->base + L.ptab_zt, pz.data(), sizeof(double) * pz.size(), cudaMemcpyHostToDevice, ctx->st));
        CK(cudaStreamSynchronize(ctx->st));
        z.ptab = (const double *)(ctx->base + L.ptab_zt);
        // halo slices and exchange buffers start from zeros (they are read by passes that run over whole arrays)
        CK(cudaMemsetAsync(ctx->base, 0, L.partials, ctx->st));
        CK(cudaMemsetAsync(ctx->base + L.xbuf[0], 0, L.ptab_zt - L.xbuf[0], ctx->st));
    }
    CK(cudaMemsetAsync(s.partials, 0, L.ctrl - L.partials, ctx->st));   // the group tickets of the two-level reduction start at zero
    CK(cudaMemsetAsync(s.ctrl, 0, sizeof(Ctrl), ctx->st));
    CK(cudaMemsetAsync(s.hist, 0, sizeof(double2) * LGF_HIST_CAP, ctx->st));
    CK(cudaStreamSynchronize(ctx->st)); // the host vectors above go out of scope
    ctx->tiled = (ctx->fft_path == 0) && fft_tiled_supported(ctx->N, ctx->prec);
    if (ctx->tiled && fft_tiled_setup(ctx->N, ctx->prec) != 0) {
        cudaError_t e = cudaGetLastError();
        return cuda_fail(ctx, e, "fft_tiled_setup");
    }
    ctx->use_gbuf = ctx->fusion && ctx->tiled && ctx->pack == 4 && ctx->fft_passes != 8 && fft_tiled_gbuf_supported(ctx->N, ctx->prec);
    l2_window_clear(ctx);
    if (ctx->use_gbuf) l2_window_set(ctx);   // one field buffer, used in place by every pass
    graph_drop(ctx);
    ctx->acc_dirty = false;
    ctx->bound = true;
    ctx->loaded = false;
    ctx->wstate = 0;
    return LGF_OK;
}

int lgf_load_links(lgf_ctx *ctx, const void *src, int src_is_device, int src_layout)
{
    if (!ctx) return LGF_ERR_INVALID_ARG;
    if (!ctx->bound) return fail(ctx, LGF_ERR_NOT_BOUND, "lgf_bind has not been called");
    if (!src) return fail(ctx, LGF_ERR_INVALID_ARG, "src is NULL");
    if (src_layout != LGF_LAYOUT_AOS && src_layout != LGF_LAYOUT_AOS12) return fail(ctx, LGF_ERR_INVALID_ARG, "unknown layout");
    const int per = src_layout == LGF_LAYOUT_AOS12 ? 6 : 9;
    const size_t e = elem_bytes(ctx);
    if (src_is_device) {
        run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_aos_to_soa(ctx->sa, src, per, 0, ctx->V, ctx->st); });
    } else {
        char *stg = ctx->base + ctx->lay.staging;
        for (int64_t s0 = 0; s0 < ctx->V; s0 += ctx->lay.staging_sites) {
            const int64_t n = std::min<int64_t>(ctx->lay.staging_sites, ctx->V - s0);
            CK(cudaMemcpyAsync(stg, (const char *)src + (size_t)s0 * 4 * per * e, (size_t)n * 4 * per * e, cudaMemcpyHostToDevice, ctx->st));
            run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_aos_to_soa(ctx->sa, stg, per, s0, n, ctx->st); });
        }
    }
    if (ctx->accum) {
        run_kernel(ctx, LGF_KERNEL_APPLY_G, 1, [&] { launch_g_identity(ctx->sa, ctx->gbuf, ctx->st); });
        ctx->acc_dirty = false;
    }
    int rc = clear_done(ctx);
    if (rc) return rc;
    if (ctx->shard_world == 0) do_measure(ctx, -1.0, 0);     // sharded: the measure needs the halo links first (lgf_shard_step)
    CK(cudaGetLastError());
    if (!src_is_device) CK(cudaStreamSynchronize(ctx->st));
    ctx->loaded = true;
    return LGF_OK;
}

int lgf_get_links(lgf_ctx *ctx, void *dst, int dst_is_device, int dst_layout)
{
    int rc = need_loaded(ctx);
    if (rc) return rc;
    if (!dst) return fail(ctx, LGF_ERR_INVALID_ARG, "dst is NULL");
    if (dst_layout != LGF_LAYOUT_AOS && dst_layout != LGF_LAYOUT_AOS12) return fail(ctx, LGF_ERR_INVALID_ARG, "unknown layout");
    const int per = dst_layout == LGF_LAYOUT_AOS12 ? 6 : 9;
    materialise(ctx);
    const size_t e = elem_bytes(ctx);
    if (dst_is_device) {
        run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_soa_to_aos(ctx->sa, dst, per, 0, ctx->V, ctx->st); });
    } else {
        char *stg = ctx->base + ctx->lay.staging;
        for (int64_t s0 = 0; s0 < ctx->V; s0 += ctx->lay.staging_sites) {
            const int64_t n = std::min<int64_t>(ctx->lay.staging_sites, ctx->V - s0);
            run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_soa_to_aos(ctx->sa, stg, per, s0, n, ctx->st); });
            CK(cudaMemcpyAsync((char *)dst + (size_t)s0 * 4 * per * e, stg, (size_t)n * 4 * per * e, cudaMemcpyDeviceToHost, ctx->st));
        }
    }
    CK(cudaStreamSynchronize(ctx->st));
    CK(cudaGetLastError());
    return LGF_OK;
}

int lgf_measure(lgf_ctx *ctx, double *F, double *theta)
{
    int rc = need_unsharded(ctx);
    if (rc) return rc;
    if ((rc = clear_done(ctx))) return rc;
    materialise(ctx);
    do_measure(ctx, -1.0, 0);
    Ctrl h;
    if ((rc = read_ctrl(ctx, &h))) return rc;
    if (F) *F = h.F;
    if (theta) *theta = h.theta;
    return LGF_OK;
}

int lgf_iterate(lgf_ctx *ctx, double alpha, int64_t n, lgf_result *out)
{
    int rc = need_unsharded(ctx);
    if (rc) return rc;
    if (n < 0) return fail(ctx, LGF_ERR_INVALID_ARG, "n must be >= 0");
    if (ctx->wstate != 1) {
        if ((rc = clear_done(ctx))) return rc;
        materialise(ctx);
        do_measure(ctx, -1.0, 0);
    }
    run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_ctrl_reset(ctx->sa, -1.0, ctx->st); });
    const int cur0 = ctx->cur, wcur0 = ctx->wcur;
    run_iterations(ctx, alpha, -1.0, n);
    CK(cudaGetLastError());
    if (out) {
        Ctrl h;
        if ((rc = read_ctrl(ctx, &h))) return rc;
        settle_buffers(ctx, cur0, wcur0, h.iter);
        out->iterations = h.iter; out->F = h.F; out->theta = h.theta; out->converged = 0;
        if (h.done == 2) return fail(ctx, LGF_ERR_NUMERIC, "theta is NaN or Inf");
    }
    return LGF_OK;
}

int lgf_fix(lgf_ctx *ctx, double alpha, double eps, lgf_result *out)
{
    int rc = need_unsharded(ctx);
    if (rc) return rc;
    if (!(eps >= 0)) return fail(ctx, LGF_ERR_INVALID_ARG, "eps must be >= 0");
    if (ctx->wstate != 1) {
        if ((rc = clear_done(ctx))) return rc;
        materialise(ctx);
        do_measure(ctx, -1.0, 0);
    }
    run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_ctrl_reset(ctx->sa, eps, ctx->st); });
    Ctrl h;
    if ((rc = read_ctrl(ctx, &h))) return rc;
    int64_t launched = 0;
    const int cur0 = ctx->cur, wcur0 = ctx->wcur;
    while (!h.done && launched < ctx->max_iter) {
        const int64_t n = std::min<int64_t>(ctx->check_interval, ctx->max_iter - launched);
        run_iterations(ctx, alpha, eps, n);
        launched += n;
        CK(cudaGetLastError());
        if ((rc = read_ctrl(ctx, &h))) return rc;
    }
    settle_buffers(ctx, cur0, wcur0, h.iter);
    ctx->wstate = 1; // kernels after `done` exited at once: w still holds Delta of the final links
    if (out) { out->iterations = h.iter; out->F = h.F; out->theta = h.theta; out->converged = (h.done == 1); }
    if (h.done == 2) return fail(ctx, LGF_ERR_NUMERIC, "theta is NaN or Inf");
    if (!h.done) return fail(ctx, LGF_ERR_NOT_CONVERGED, "MAX_ITER reached before theta <= eps");
    return LGF_OK;
}

int lgf_stage(lgf_ctx *ctx, int stage, double alpha)
{
    int rc = need_unsharded(ctx);
    if (rc) return rc;
    if ((rc = clear_done(ctx))) return rc;
    materialise(ctx);
    switch (stage) {
    case LGF_STAGE_MEASURE: do_measure(ctx, -1.0, 0); break;
    case LGF_STAGE_FOURIER:
        if (ctx->wstate != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "FOURIER needs Delta in the field buffer (run MEASURE or set DELTA)");
        do_fourier(ctx); break;
    case LGF_STAGE_UPDATE:
        if (ctx->wstate != 2) return fail(ctx, LGF_ERR_INVALID_ARG, "UPDATE needs w in the field buffer (run FOURIER or set W)");
        do_update(ctx, alpha); break;
    default: return fail(ctx, LGF_ERR_INVALID_ARG, "unknown stage");
    }
    CK(cudaStreamSynchronize(ctx->st));
    CK(cudaGetLastError());
    return LGF_OK;
}

int lgf_get_field(lgf_ctx *ctx, int which, double alpha, void *dst, int dst_is_device)
{
    int rc = need_loaded(ctx);
    if (rc) return rc;
    if (!dst) return fail(ctx, LGF_ERR_INVALID_ARG, "dst is NULL");
    if (which == LGF_FIELD_DELTA) { if (ctx->wstate != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "field buffer does not hold Delta"); }
    else if (which == LGF_FIELD_W || which == LGF_FIELD_G) { if (ctx->wstate != 2) return fail(ctx, LGF_ERR_INVALID_ARG, "field buffer does not hold w"); }
    else return fail(ctx, LGF_ERR_INVALID_ARG, "unknown field");
    const size_t e = elem_bytes(ctx);
    if (dst_is_device) {
        run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_field_get(ctx->sa, which, alpha, dst, 0, ctx->V, ctx->st); });
    } else {
        char *stg = ctx->base + ctx->lay.staging;
        for (int64_t s0 = 0; s0 < ctx->V; s0 += ctx->lay.staging_sites) {
            const int64_t n = std::min<int64_t>(ctx->lay.staging_sites, ctx->V - s0);
            run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_field_get(ctx->sa, which, alpha, stg, s0, n, ctx->st); });
            CK(cudaMemcpyAsync((char *)dst + (size_t)s0 * 9 * e, stg, (size_t)n * 9 * e, cudaMemcpyDeviceToHost, ctx->st));
        }
    }
    CK(cudaStreamSynchronize(ctx->st));
    CK(cudaGetLastError());
    return LGF_OK;
}

int lgf_set_field(lgf_ctx *ctx, int which, const void *src, int src_is_device)
{
    int rc = need_loaded(ctx);
    if (rc) return rc;
    if (!src) return fail(ctx, LGF_ERR_INVALID_ARG, "src is NULL");
    if (which != LGF_FIELD_DELTA && which != LGF_FIELD_W) return fail(ctx, LGF_ERR_INVALID_ARG, "only DELTA and W can be set");
    materialise(ctx);
    const size_t e = elem_bytes(ctx);
    if (src_is_device) {
        run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_field_set(ctx->sa, src, 0, ctx->V, ctx->st); });
    } else {
        char *stg = ctx->base + ctx->lay.staging;
        for (int64_t s0 = 0; s0 < ctx->V; s0 += ctx->lay.staging_sites) {
            const int64_t n = std::min<int64_t>(ctx->lay.staging_sites, ctx->V - s0);
            CK(cudaMemcpyAsync(stg, (const char *)src + (size_t)s0 * 9 * e, (size_t)n * 9 * e, cudaMemcpyHostToDevice, ctx->st));
            run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_field_set(ctx->sa, stg, s0, n, ctx->st); });
        }
    }
    CK(cudaStreamSynchronize(ctx->st));
    CK(cudaGetLastError());
    ctx->wstate = (which == LGF_FIELD_DELTA) ? 1 : 2;
    return LGF_OK;
}

int lgf_history(lgf_ctx *ctx, double *F, double *theta, int cap, int *n)
{
    int rc = need_loaded(ctx);
    if (rc) return rc;
    if (!n || cap < 0) return fail(ctx, LGF_ERR_INVALID_ARG, "bad arguments");
    Ctrl h;
    if ((rc = read_ctrl(ctx, &h))) return rc;
    int64_t cnt = h.iter + 1;
    if (cnt > LGF_HIST_CAP) cnt = LGF_HIST_CAP;
    if (cnt > cap) cnt = cap;
    std::vector<double2> tmp((size_t)cnt);
    if (cnt) {
        CK(cudaMemcpyAsync(tmp.data(), ctx->sa.hist, sizeof(double2) * (size_t)cnt, cudaMemcpyDeviceToHost, ctx->st));
        CK(cudaStreamSynchronize(ctx->st));
    }
    for (int64_t i = 0; i < cnt; i++) {
        if (F) F[i] = tmp[(size_t)i].x;
        if (theta) theta[i] = tmp[(size_t)i].y;
    }
    *n = (int)cnt;
    return LGF_OK;
}

int lgf_kernel_time(lgf_ctx *ctx, int kind, double *ms, int64_t *launches)
{
    if (!ctx) return LGF_ERR_INVALID_ARG;
    if (kind < 0 || kind >= LGF_KERNEL_KINDS) return fail(ctx, LGF_ERR_INVALID_ARG, "unknown kernel kind");
    if (ctx->bound) flush_events(ctx);
    if (ms) *ms = ctx->kms[kind];
    if (launches) *launches = ctx->kcount[kind];
    return LGF_OK;
}

int64_t lgf_launch_count(const lgf_ctx *ctx) { return ctx ? ctx->launches : 0; }

int lgf_reset_counters(lgf_ctx *ctx)
{
    if (!ctx) return LGF_ERR_INVALID_ARG;
    if (ctx->bound) flush_events(ctx);
    ctx->launches = 0;
    for (int k = 0; k < LGF_KERNEL_KINDS; k++) { ctx->kms[k] = 0; ctx->kcount[k] = 0; }
    return LGF_OK;
}

int lgf_uses_tiled_fft(const lgf_ctx *ctx) { return ctx && ctx->tiled ? 1 : 0; }
int lgf_uses_gbuf(const lgf_ctx *ctx) { return ctx && ctx->bound && ctx->use_gbuf ? 1 : 0; }
int lgf_zblock(const lgf_ctx *ctx) { return ctx && ctx->bound ? ctx->sa.geo.zb : 0; }

int lgf_shard_step(lgf_ctx *ctx, int step, double alpha, double eps)
{
    int rc = need_loaded(ctx);
    if (rc) return rc;
    if (ctx->shard_world <= 0) return fail(ctx, LGF_ERR_INVALID_ARG, "not a sharded context (LGF_OPT_SHARD_WORLD)");
    switch (step) {
    case LGF_SHARD_MEASURE:
        if ((rc = clear_done(ctx))) return rc;
        do_measure(ctx, -1.0, 0); break;
    case LGF_SHARD_RESET:
        run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_ctrl_reset(ctx->sa, eps, ctx->st); }); break;
    case LGF_SHARD_XY_FWD:
        if (ctx->wstate != 1) return fail(ctx, LGF_ERR_INVALID_ARG, "XY_FWD needs Delta in the field buffer");
        run_kernel(ctx, LGF_KERNEL_FFT_XY_FWD, 1, [&] { launch_fft_tiled(ctx->fa, 0, ctx->st); }); break;
    case LGF_SHARD_PACK:
        run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_slab_pack(ctx->sa, ctx->xbuf[0], ctx->shard_world, 0, ctx->st); }); break;
    case LGF_SHARD_ZT:
        run_kernel(ctx, LGF_KERNEL_FFT_ZT, 1, [&] { launch_fft_tiled(ctx->fa_zt, 1, ctx->st); }); break;
    case LGF_SHARD_UNPACK:
        run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_slab_pack(ctx->sa, ctx->xbuf[0], ctx->shard_world, 1, ctx->st); }); break;
    case LGF_SHARD_XY_INV_G:
        run_kernel(ctx, LGF_KERNEL_FFT_XY_INV_G, 1, [&] { launch_fft_tiled_inv_g(ctx->fa, ctx->gbuf, alpha, ctx->gmap, 0, ctx->st); });
        ctx->wstate = 2; break;
    case LGF_SHARD_LINK: {
        void *lin = ctx->links_buf[ctx->cur], *lout = ctx->links_buf[ctx->cur ^ 1];
        run_kernel(ctx, LGF_KERNEL_UPDATE_MEASURE, 1,
                   [&] { launch_update_measure(ctx->sa, lin, lout, ctx->gbuf, 1, ctx->w_buf[ctx->wcur], alpha, -1.0, ctx->st); });
        ctx->cur ^= 1;
        sync_ptrs(ctx);
        ctx->wstate = 1;
        break;
    }
    case LGF_SHARD_FINISH:
        run_kernel(ctx, LGF_KERNEL_LAYOUT, 1, [&] { launch_slab_finish(ctx->sa, eps, ctx->st); }); break;
    default: return fail(ctx, LGF_ERR_INVALID_ARG, "unknown shard step");
    }
    CK(cudaGetLastError());
    return LGF_OK;
}

int lgf_shard_region(const lgf_ctx *ctx, int region, size_t *offset, size_t *bytes)
{
    if (!ctx || !ctx->bound || ctx->shard_world <= 0 || !offset || !bytes) return LGF_ERR_INVALID_ARG;
    const size_t e = ctx->prec == LGF_PREC_FP64 ? 16 : 8;
    const int ne = ctx->recon == 12 ? 6 : 9;
    const Layout &L = ctx->lay;
    switch (region) {
    case LGF_REGION_CTRL: *offset = L.ctrl; *bytes = 2 * sizeof(double); break;        /* F, theta: the first two doubles */
    case LGF_REGION_XSEND: *offset = L.xbuf[0]; *bytes = (size_t)4 * ctx->V * e; break;
    case LGF_REGION_XRECV: *offset = L.xbuf[1]; *bytes = (size_t)4 * ctx->V * e; break;
    case LGF_REGION_G: *offset = L.gbuf; *bytes = (size_t)6 * ctx->Vp * e; break;
    case LGF_REGION_LINKS: *offset = L.links[ctx->cur]; *bytes = (size_t)4 * ne * ctx->Vp * e; break;
    default: return LGF_ERR_INVALID_ARG;
    }
    return LGF_OK;
}

int lgf_shard_info(const lgf_ctx *ctx, int64_t *info, int n)
{
    if (!ctx || !ctx->bound || ctx->shard_world <= 0 || !info || n < 8) return LGF_ERR_INVALID_ARG;
    info[0] = ctx->Vp;                                                   /* stored sites per array (with halos) */
    info[1] = (int64_t)ctx->N[0] * ctx->N[1] * ctx->N[2];                /* sites of one time slice */
    info[2] = ctx->N[3] / ctx->shard_world;                              /* own time slices */
    info[3] = ctx->recon == 12 ? 6 : 9;                                  /* complex arrays per link direction */
    info[4] = ctx->prec == LGF_PREC_FP64 ? 16 : 8;                       /* bytes per complex number */
    info[5] = ctx->shard_world; info[6] = ctx->shard_rank; info[7] = ctx->V;
    return LGF_OK;
}

int lgf_shard_result(lgf_ctx *ctx, lgf_result *out)
{
    int rc = need_loaded(ctx);
    if (rc) return rc;
    if (!out) return fail(ctx, LGF_ERR_INVALID_ARG, "out is NULL");
    Ctrl h;
    if ((rc = read_ctrl(ctx, &h))) return rc;
    out->iterations = h.iter; out->F = h.F; out->theta = h.theta; out->converged = (h.done == 1);
    if (h.done == 2) return fail(ctx, LGF_ERR_NUMERIC, "theta is NaN or Inf");
    return LGF_OK;
}

int lgf_sync_links(lgf_ctx *ctx)
{
    int rc = need_loaded(ctx);
    if (rc) return rc;
    materialise(ctx);
    CK(cudaGetLastError());
    return LGF_OK;
}

const char *lgf_last_error(const lgf_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

int lgf_destroy(lgf_ctx *ctx)
{
    if (!ctx) return LGF_OK;
    l2_window_clear(ctx);
    graph_drop(ctx);
    for (auto &p : ctx->evs) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
    delete ctx;
    return LGF_OK;
}

} // extern "C"
