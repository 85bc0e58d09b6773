/*
 * lgf.h -- C ABI of liblgf.so: Fourier-accelerated steepest-descent SU(3) Landau gauge
 * fixing on a periodic 4D lattice (arXiv 1210.8018, Algorithm 1), on one
 * NVIDIA B200 (sm_100a).
 *
 * Conventions
 *   - Every function returns an int status: LGF_OK (0) or a negative LGF_ERR_* code.  No
 *     exception, exit() or abort() crosses this boundary.  lgf_last_error(ctx) gives text.
 *   - "host" / "device" is stated for every pointer.  Device pointers are plain CUDA device
 *     addresses on the current device; the library never takes ownership of a caller buffer.
 *   - The library allocates no device memory: the caller (PyTorch in this repo) hands it ONE
 *     device workspace of lgf_workspace_bytes() bytes and a CUDA stream with lgf_bind().
 *   - Not thread-safe per context; distinct contexts are independent.
 *
 * Lattice and layouts
 *   extents N[0..3] = Nx, Ny, Nz, Nt;  V = Nx*Ny*Nz*Nt;  direction mu = 0..3 <-> x, y, z, t;
 *   site index s = ix + Nx*(iy + Ny*(iz + Nz*it))  (x fastest, lexicographic).
 *   Interchange layouts of a link field:
 *     LGF_LAYOUT_AOS:    real[((((s*4 + mu)*3 + row)*3 + col)*2 + {0:re, 1:im}],   18 reals per link,
 *     LGF_LAYOUT_AOS12:  the same with row = 0, 1 only, real[((((s*4 + mu)*2 + row)*3 + col)*2 + {re,im}],
 *                        12 reals per link (the 12-real compression of PAPER.md:121-123 as an exchange
 *                        format: two thirds of the bytes over PCIe); row 2 = conj(row0 x row1) is
 *                        implied, and rebuilt on load when the context stores 18 reals,
 *   and of a site field (Delta, w, g):  real[(((s*3 + row)*3 + col)*2 + {re,im}].
 *   `real` is double for LGF_PREC_FP64 contexts and float for LGF_PREC_FP32 contexts.
 *   Inside the workspace links live as complex SoA arrays (one array over sites per matrix
 *   element), 9 or 6 elements per link (12-real compression).
 */
#ifndef LGF_H
#define LGF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lgf_ctx lgf_ctx;

/* Result of lgf_iterate / lgf_fix.  F and theta are those of the final links. */
typedef struct lgf_result {
    int64_t iterations; /* executions of the loop body of Algorithm 1 (= link updates) in this call */
    double F;           /* eq. 1.1 at g = 1 on the current links */
    double theta;       /* eq. 1.4 */
    int converged;      /* 1 if theta <= eps was reached (lgf_fix), else 0 */
} lgf_result;

enum {
    LGF_OK = 0,
    LGF_ERR_INVALID_ARG = -1,
    LGF_ERR_UNSUPPORTED_SIZE = -2,
    LGF_ERR_NOT_BOUND = -3,
    LGF_ERR_NOT_LOADED = -4,
    LGF_ERR_WORKSPACE_TOO_SMALL = -5,
    LGF_ERR_CUDA = -6,
    LGF_ERR_NOT_CONVERGED = -7,
    LGF_ERR_NUMERIC = -8
};

enum { LGF_PREC_FP64 = 0, LGF_PREC_FP32 = 1 };
enum { LGF_LAYOUT_AOS = 0, LGF_LAYOUT_AOS12 = 1 };

/* lgf_set_option keys.  Options must be set before lgf_workspace_bytes / lgf_bind. */
enum {
    LGF_OPT_RECON = 1,          /* 18 (default) or 12 reals stored per link.  The links handed
                                   to lgf_load_links must be SU(3) to working precision either way: with 12 reals
                                   row 2 is never stored, and with 18 reals the fused link kernel (FUSION = 1)
                                   stores row 2 of g U g^dagger as conj(row0 x row1) of the product instead of
                                   multiplying it out (equal to rounding for special unitary links, DESIGN.md
                                   reading R15); FUSION = 0 multiplies all three rows. */
    LGF_OPT_FFT_BATCH = 2,      /* 4 (default): Delta packed into 4 complex fields; 9: one FFT per
                                   element of the Delta matrix as in Alg. 1 line 3 */
    LGF_OPT_MAX_ITER = 3,       /* iteration cap of lgf_fix, default 100000 */
    LGF_OPT_CHECK_INTERVAL = 4, /* iterations launched between two host polls of the device
                                   `done` flag in lgf_fix, default 8.  Does not change results:
                                   kernels launched after convergence exit at once. */
    LGF_OPT_FFT_PATH = 5,       /* 0 (default): tiled register FFT when the extents allow it,
                                   1: always the generic per-axis transform */
    LGF_OPT_PROFILE = 6,        /* 1: bracket every kernel launch with CUDA events on the bound
                                   stream so that lgf_kernel_time works; default 0 */
    LGF_OPT_FUSION = 7,         /* 1 (default): lgf_iterate / lgf_fix run the link update and the
                                   measure of the next iteration as ONE kernel over double-buffered
                                   links (each link read once, written once per iteration), with g
                                   built in the last FFT pass where the tile fits;
                                   0: the three separate kernels of lgf_stage (measure, Fourier,
                                   update in place), as in the paper's kernel list */
    LGF_OPT_L2_PERSIST = 8,     /* 1: when the field buffer (Delta / w) fits in the persisting part of the
                                   L2 cache, lgf_bind sets an access-policy window on the bound stream so
                                   that the passes over the field between the link kernels are served by
                                   L2 instead of HBM (sets the device limit cudaLimitPersistingL2CacheSize;
                                   undone by lgf_destroy).  0 (default): off -- measured slower at 32^4,
                                   the set-aside takes L2 away from the link kernel's neighbour re-reads
                                   (DESIGN.md section 6). */
    LGF_OPT_GMAP = 9,           /* how g(x) is formed from w(x).  0 (default): the paper's choice, first
                                   order g = 1 + (alpha/2) w followed by a reunitarisation;
                                   1: the exact exponential g = exp((alpha/2) w) of eq. 1.2 as written
                                   (PAPER.md:49), no projection.  May be changed at any time. */
    LGF_OPT_ACCUM_G = 10,       /* 1: lgf_iterate / lgf_fix keep the loaded links fixed and accumulate the
                                   gauge transformation instead, G(x) <- g(x) G(x) (rows 0, 1 stored, Gram-
                                   Schmidt after every product), measuring Delta, F, theta of
                                   G(x) U_mu(x) G^dagger(x+mu) on the fly; the links are rewritten once,
                                   when an iterate / fix call returns control to any other call that needs
                                   them (lgf_get_links, lgf_measure, lgf_stage, field taps).  The same
                                   iteration as Alg. 1 lines 12-16 up to rounding, without the
                                   per-iteration link write; one link buffer instead of two.  Needs FUSION = 1,
                                   FFT_BATCH = 4 and a lattice the tiled FFT covers, else lgf_bind fails with
                                   LGF_ERR_INVALID_ARG.  0 (default): links rewritten every iteration. */
    LGF_OPT_GRAPH = 11,         /* 1 (default): lgf_iterate / lgf_fix capture min(CHECK_INTERVAL, 8) (rounded
                                   down to even, at least 2) iterations into a CUDA graph and replay it, so
                                   that small lattices (8^4, 16^4: a few microseconds per kernel) are not
                                   bound by launch overhead.  The first batch with given (alpha, eps) is
                                   launched directly and the graph captured behind it (host work hidden by
                                   the running kernels); later batches and later calls replay it.  Leftovers
                                   and profiled runs (LGF_OPT_PROFILE) are launched directly.  Same kernels, same results.  Falls back to direct
                                   launches by itself when the bound stream cannot be captured (e.g. the
                                   legacy default stream).  0: always direct launches.  Any time. */
    LGF_OPT_ZBLOCK = 12,        /* order in which the per-site kernels (measure, update, fused link kernel) walk
                                   the lattice: the (z,t) planes are visited in blocks of ZBLOCK consecutive z,
                                   all Nt time slices of a z-block before the next one, so that the -mu / +mu
                                   neighbours of a site (Alg. 1 lines 12-16) were touched a few
                                   planes ago and are still in L2 even when one time slice of links is larger
                                   than L2 (64^4).  0 (default): chosen by lgf_bind from the L2 size of the device
                                   (the largest divisor of Nz whose block of planes takes at most about a third
                                   of L2); a positive value must divide Nz (Nz = plain storage order).  Changes
                                   only the order of the FP64 partial sums of F and theta (1e-16 relative), not
                                   what is computed.  Before lgf_bind. */
    LGF_OPT_ZT_PIPE = 13,       /* middle pass of the tiled FFT ((z,t) forward, mask, (z,t) inverse; Alg. 1 lines 3-8,
                                   PAPER.md:80-90).  1: persistent CTAs that keep their shared-memory tile and fetch
                                   the next tile with asynchronous copies (cp.async) while the current one is
                                   finished; 0: one tile per thread group, loaded straight into registers.  Same
                                   arithmetic in the same order: bitwise the same w.  Any time. */
    LGF_OPT_FFT_PASSES = 14,    /* pass structure of the tiled 4D FFT, the axis of the paper's comparison of 4 x 1D,
                                   2D + 2D and 3D + 1D decompositions.  3 (default): (x,y) forward |
                                   (z,t) forward, mask, (z,t) inverse in one tile visit | (x,y) inverse.  4: 2D + 2D
                                   as the paper runs it, (x,y) forward | (z,t) forward and mask | (z,t) inverse |
                                   (x,y) inverse (available for square and 32 x n (z,t) tiles).  8: 4 x 1D, one pass per
                                   axis and direction with the same register lines (g is then rebuilt from w by the link
                                   kernel; not with ACCUM_G).  Same w to rounding; timing comparison only
                                   (bench_sweep.py --passes).  lgf_bind fails with LGF_ERR_INVALID_ARG where a structure
                                   is not available.  Before lgf_bind. */
    LGF_OPT_SHARD_WORLD = 15,   /* R > 0: this context holds ONE t-slab of a lattice sharded over R GPUs (the B200
                                   analogue of the paper's distributed CPU program):
                                   lgf_create was given the extents of the WHOLE lattice, the context stores the
                                   Nt / R time slices of rank SHARD_RANK between one halo slice below and one
                                   above, and lgf_load_links / lgf_get_links move those Nt / R slices
                                   ([Nx Ny Nz Nt/R] sites, same interchange layouts).  R must divide Nt and Ny.
                                   The iteration is then driven step by step with lgf_shard_step, the exchanges
                                   between the steps (all-to-all transposes of the packed field around the (z,t)
                                   pass, one-slice halos of g and of the t-links, the all-reduce of F and theta)
                                   being the caller's (paper_1210_8018_b200/sharded.py: torch.distributed over NCCL).
                                   R = 1 is valid (the exchanges are with itself).  Default path only (FUSION = 1,
                                   FFT_BATCH = 4, FFT_PASSES = 3, no ACCUM_G, tiled FFT).  0 (default): off.
                                   Before lgf_bind. */
    LGF_OPT_SHARD_RANK = 16,    /* which slab, 0 <= rank < SHARD_WORLD: time slices [rank Nt/R, (rank+1) Nt/R).
                                   Set after SHARD_WORLD, before lgf_bind. */
    LGF_OPT_TMARCH = 17,        /* 0 (default: 4 for FP32 contexts without ACCUM_G, else 1, as measured), 1, 2 or 4:
                                   consecutive time slices a thread of the fused link kernel walks.  From its
                                   second site on the -t neighbour is the thread's own previous site, whose product
                                   g(x) U_t(x) it has just formed (Alg. 1 lines 12-16), so 12 of the
                                   102 loads and one of the nine 3x3 products per site are saved.  Falls back to 1
                                   when it does not divide the number of time slices the context walks.  Same
                                   arithmetic per link; the order of the F, theta partial sums changes (1e-16).
                                   Before lgf_bind. */
    LGF_OPT_LINK_TILE = 18,     /* the fused link kernel on 4D tiles: 0 (default) or 1 = off (one thread per site in
                                   walk order, k_update_measure), 128 / 256 / 512 = threads (sites) per tile.  A CTA
                                   owns an Nx x TDy x TDz x TDt tile; each thread forms its four new links
                                   U'_mu(x) = g(x) U_mu(x) g^dagger(x+mu) once (Alg. 1 lines 12-16) and
                                   hands the anti-Hermitian part of each, which is all that Delta(x+mu) needs of it
                                   (eq. 1.5), to the thread of x+mu through shared memory; only backward
                                   links across a tile face are rebuilt from the old links.  Same links bit for bit;
                                   Delta, F, theta differ in the order of their sums (1e-16).  Measured slower than
                                   the site kernel on B200 (profiles/r02_link_tile.md), hence off by default.
                                   Ignored (site kernel) for sharded contexts, with ACCUM_G, with FUSION = 0 and when
                                   Nx exceeds the tile.  Takes precedence over TMARCH.  Before lgf_bind. */
    LGF_OPT_LINK_STREAM = 19    /* 1: the fused link kernel as a stream (k_update_measure_stream).  Persistent CTAs
                                   walk tiles of 128 consecutive sites; a producer warp fetches the tile's own links
                                   U_mu(x), the 4 x 6 or 4 x 9 SoA lines per site that must come from DRAM (Alg. 1
                                   lines 12-16), with cp.async.bulk (the TMA engine) into a ring of
                                   shared-memory stages, completion on an mbarrier, while four consumer warps do the
                                   arithmetic of the previous tile.  Same links bit for bit; F and theta are summed
                                   per CTA over its tiles (order of the sums only).  Needs the default path (FUSION = 1,
                                   FFT_BATCH = 4, tiled FFT: the g buffer) and Nx Ny divisible by 128; ignored
                                   otherwise, for sharded contexts and with ACCUM_G.  Takes precedence over LINK_TILE
                                   and TMARCH.  0 (default): off.  Before lgf_bind. */
};

/* lgf_shard_step selectors: the kernels of one iteration of a sharded lattice, in the order of a step
 * (exchanges the caller performs are in brackets):
 *   start:      [halo of the t-links]  MEASURE  [all-reduce F, theta]  RESET
 *   iteration:  XY_FWD  PACK  [all-to-all send -> recv]  ZT  [all-to-all recv -> send]  UNPACK  XY_INV_G
 *               [halos of g]  LINK  [halo of the new t-links]  [all-reduce F, theta]  FINISH */
enum {
    LGF_SHARD_MEASURE = 0,   /* kernel (a) on the slab: Delta, and this rank's part of F and theta */
    LGF_SHARD_RESET = 1,     /* after the all-reduce: iteration counter 0, history[0], done = (theta <= eps) */
    LGF_SHARD_XY_FWD = 2,    /* (x,y) forward pass of the FFT on the slab */
    LGF_SHARD_PACK = 3,      /* field -> send buffer, one contiguous block per destination rank */
    LGF_SHARD_ZT = 4,        /* (z,t) forward, mask, (z,t) inverse on the receive buffer (all t, this rank's rows of y) */
    LGF_SHARD_UNPACK = 5,    /* send buffer (after the return all-to-all) -> field */
    LGF_SHARD_XY_INV_G = 6,  /* (x,y) inverse pass and g(x) (uses alpha) */
    LGF_SHARD_LINK = 7,      /* fused link update + measure of the new links (uses alpha): this rank's part of F, theta */
    LGF_SHARD_FINISH = 8     /* after the all-reduce: history entry, done = (theta <= eps) */
};
/* lgf_shard_region selectors: byte ranges of the bound workspace that the caller exchanges */
enum {
    LGF_REGION_CTRL = 0,     /* two doubles: F, theta (all-reduce, sum) */
    LGF_REGION_XSEND = 1,    /* send buffer of the transposes: SHARD_WORLD equal contiguous blocks */
    LGF_REGION_XRECV = 2,    /* receive buffer */
    LGF_REGION_G = 3,        /* rows 0, 1 of g: 6 complex arrays of `stored sites` each, time slice t at t * slice sites */
    LGF_REGION_LINKS = 4     /* the CURRENT link buffer (changes with every LINK step): 4 x NE complex arrays of
                                `stored sites` each, array (mu * NE + k), own slices at t = 1..Nt/R, halos at 0 and Nt/R + 1 */
};

/* lgf_get_field / lgf_set_field selectors */
enum {
    LGF_FIELD_DELTA = 0, /* Delta(x) of the current links, eq. 1.5 (valid after a measure) */
    LGF_FIELD_W = 1,     /* w(x) = F^-1 (p_max^2/p^2) F Delta, normalised (valid after LGF_STAGE_FOURIER) */
    LGF_FIELD_G = 2      /* g(x) = reunit(1 + (alpha/2) w(x)) built from the current w (get only) */
};

/* lgf_stage selectors: the three kernels of one iteration, for per-kernel parity tests */
enum {
    LGF_STAGE_MEASURE = 0, /* kernel (a): Delta, F, theta from the links */
    LGF_STAGE_FOURIER = 1, /* kernel (b): Delta -> w in place (Alg. 1 lines 3-8) */
    LGF_STAGE_UPDATE = 2   /* kernel (c): g(x), U_mu(x) <- g(x) U_mu(x) g^dagger(x+mu) */
};

/* kernel kinds for lgf_kernel_time */
enum {
    LGF_KERNEL_MEASURE = 0,
    LGF_KERNEL_FFT_XY_FWD = 1,
    LGF_KERNEL_FFT_ZT = 2,
    LGF_KERNEL_FFT_XY_INV = 3,
    LGF_KERNEL_UPDATE = 4,
    LGF_KERNEL_FFT_GENERIC = 5,
    LGF_KERNEL_LAYOUT = 6,
    LGF_KERNEL_FFT_XY_INV_G = 7,   /* last FFT pass with the g build as its epilogue */
    LGF_KERNEL_UPDATE_MEASURE = 8, /* fused link update + measure */
    LGF_KERNEL_FFT_XY_INV_GACC = 9, /* last FFT pass with g build and G <- g G as its epilogue (ACCUM_G) */
    LGF_KERNEL_MEASURE_ACC = 10,    /* Delta, F, theta of G U G^dagger from the fixed links and G (ACCUM_G) */
    LGF_KERNEL_APPLY_G = 11,        /* U <- G U G^dagger in place, G <- 1 (ACCUM_G, once per call) */
    LGF_KERNEL_KINDS = 12
};

/* Create a context for an Nx*Ny*Nz*Nt lattice.  host call; allocates host memory only.
 * Each extent must be even, 4 <= N <= 64, of the form 2^a 3^b; else LGF_ERR_UNSUPPORTED_SIZE.
 * precision: LGF_PREC_FP64, or LGF_PREC_FP32 (storage, FFT and matrix arithmetic in float,
 * F and theta accumulated in double).  *out (host) receives the context. */
int lgf_create(int Nx, int Ny, int Nz, int Nt, int precision, lgf_ctx **out);

/* Set an option (see LGF_OPT_*).  Must precede lgf_bind, except MAX_ITER, CHECK_INTERVAL, PROFILE. */
int lgf_set_option(lgf_ctx *ctx, int key, int64_t value);

/* Bytes of device workspace this context needs with its current options (0 on NULL). */
size_t lgf_workspace_bytes(const lgf_ctx *ctx);

/* Hand the context its device workspace (device pointer, 256-byte aligned, owned by the
 * caller, must outlive the context's use) and the CUDA stream (a cudaStream_t passed as
 * void*, may be NULL for the default stream) on which every kernel and copy is issued.
 * Uploads the small tables (momentum tables 4 sin^2(pi k/N), twiddles). */
int lgf_bind(lgf_ctx *ctx, void *dev_workspace, size_t bytes, void *cuda_stream);

/* Load a link field in an interchange layout (LGF_LAYOUT_AOS or LGF_LAYOUT_AOS12) from host
 * (src_is_device = 0) or device memory into the internal SoA arrays (dropping row 2 if RECON = 12,
 * rebuilding it from an AOS12 source if RECON = 18), then run kernel (a) so that
 * Delta, F, theta of the loaded links are available.  The source is not retained.
 * Synchronises the stream before returning when the source is host memory. */
int lgf_load_links(lgf_ctx *ctx, const void *src, int src_is_device, int src_layout);

/* Inverse conversion into dst (host or device) in either layout, third row rebuilt if RECON = 12 and
 * the layout carries it.  Synchronous. */
int lgf_get_links(lgf_ctx *ctx, void *dst, int dst_is_device, int dst_layout);

/* Kernel (a) only: F and theta of the current links (host out pointers, may be NULL). Synchronous. */
int lgf_measure(lgf_ctx *ctx, double *F, double *theta);

/* Exactly n iterations of the loop body of Algorithm 1 with step alpha, never looking at
 * theta (timed windows).  Asynchronous on the bound stream when out == NULL; otherwise
 * synchronises and fills *out (host). */
int lgf_iterate(lgf_ctx *ctx, double alpha, int64_t n, lgf_result *out);

/* Algorithm 1: iterate while theta > eps (stop when theta <= eps).
 * out->iterations = 0 if the loaded links already satisfy theta <= eps.  When MAX_ITER is
 * reached returns LGF_ERR_NOT_CONVERGED with *out filled; NaN/Inf in theta returns
 * LGF_ERR_NUMERIC.  The stop decision is taken on the device; the host polls it every
 * CHECK_INTERVAL iterations. */
int lgf_fix(lgf_ctx *ctx, double alpha, double eps, lgf_result *out);

/* Run one kernel of the iteration (per-kernel parity).  alpha is used by LGF_STAGE_UPDATE only. */
int lgf_stage(lgf_ctx *ctx, int stage, double alpha);

/* Copy a site field in the interchange layout ([V][3][3] complex of the context's precision)
 * out of / into the context.  LGF_FIELD_G needs alpha (ignored otherwise).  Synchronous. */
int lgf_get_field(lgf_ctx *ctx, int which, double alpha, void *dst, int dst_is_device);
int lgf_set_field(lgf_ctx *ctx, int which, const void *src, int src_is_device);

/* (F, theta) after the initial measure and after each iteration of the last lgf_fix /
 * lgf_iterate call: up to cap pairs into host arrays F[], theta[]; *n (host) = pairs written.
 * The device keeps the first LGF_HISTORY_CAP = 4096 pairs of a call only (iterations 0..4095): a run
 * that takes more iterations (MAX_ITER defaults to 100000) returns the truncated prefix, *n <= 4096,
 * while lgf_result still carries the true iteration count and the final F, theta. */
#define LGF_HISTORY_CAP 4096
int lgf_history(lgf_ctx *ctx, double *F, double *theta, int cap, int *n);

/* With LGF_OPT_PROFILE = 1: total milliseconds and launch count of one kernel kind since
 * the last lgf_reset_counters, from CUDA events on the bound stream.  Synchronises. */
int lgf_kernel_time(lgf_ctx *ctx, int kind, double *ms, int64_t *launches);
/* Kernel launches issued by this context since the last reset (always counted). */
int64_t lgf_launch_count(const lgf_ctx *ctx);
int lgf_reset_counters(lgf_ctx *ctx);

/* 1 if this context takes the tiled register-FFT path, 0 if the generic one. */
int lgf_uses_tiled_fft(const lgf_ctx *ctx);
/* 1 if the last FFT pass builds g(x) in its epilogue (fused path, 4 packed fields, plane fits in
 * shared memory of one SM or of a 2-CTA cluster), 0 if g is rebuilt from w by the link kernel.
 * Valid after lgf_bind. */
int lgf_uses_gbuf(const lgf_ctx *ctx);
/* The z-block of the site walk in use (LGF_OPT_ZBLOCK after lgf_bind resolved 0 = auto); 0 before lgf_bind. */
int lgf_zblock(const lgf_ctx *ctx);

/* LGF_OPT_ACCUM_G: bring the link buffer up to date now, U_mu(x) <- G(x) U_mu(x) G^dagger(x+mu), G <- 1
 * (two launches on the bound stream, asynchronous; the calls that read the links do this
 * themselves).  No-op, LGF_OK, when nothing is pending or ACCUM_G is off.  Needs loaded links. */
int lgf_sync_links(lgf_ctx *ctx);

/* Sharded lattice (LGF_OPT_SHARD_WORLD): run one kernel step of the iteration on this rank's slab, asynchronously on the
 * bound stream (alpha is used by XY_INV_G and LINK, eps by RESET and FINISH).  The exchanges between the steps are the
 * caller's; see the LGF_SHARD_* list for the order.  LGF_ERR_INVALID_ARG on an unsharded context. */
int lgf_shard_step(lgf_ctx *ctx, int step, double alpha, double eps);
/* Byte range (offset from the bound workspace pointer, length) of an exchanged region; host out pointers. */
int lgf_shard_region(const lgf_ctx *ctx, int region, size_t *offset, size_t *bytes);
/* info[0..7] (host): stored sites per array, sites per time slice, own time slices, complex arrays per link direction,
 * bytes per complex number, SHARD_WORLD, SHARD_RANK, sites of the interchange arrays of this rank.  n >= 8. */
int lgf_shard_info(const lgf_ctx *ctx, int64_t *info, int n);
/* (iterations, F, theta, converged) as the device holds them after the last RESET / FINISH.  Synchronises. */
int lgf_shard_result(lgf_ctx *ctx, lgf_result *out);

/* Debug entry point, not on the gauge-fixing path: the measured FP64 fused-multiply-add rate of the
 * current device (DFMA per second, best of 4 timed launches of a register-only FMA kernel on the given
 * stream, a cudaStream_t passed as void*, may be NULL).  bench.py uses it as the denominator of the "alu"
 * roofline of the one kernel that is bound by FP64 arithmetic (Table 1 flop counts).
 * Allocates and frees 8 bytes of device memory; synchronises.  *dfma_per_second: host. */
int lgf_debug_dfma_rate(void *cuda_stream, double *dfma_per_second);

/* ---- The one entry point that allocates nothing (csrc/noalloc.cu) -------------------------------------------
 * For callers that cannot allocate device memory or keep a context (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): kernel (a) of Algorithm 1 on the caller's own arrays,
 *     Delta(x) (eq. 1.5),  F (eq. 1.1),  theta (eq. 1.4),
 * with the same arithmetic and the same fixed-order FP64 reduction as lgf_measure.  No context, no workspace:
 * the kernel's scratch memory (block partial sums, ticket counter, result block) is a static device array of
 * LGF_NOALLOC_SCRATCH_BYTES = 131 584 bytes that every GPU that loads the library holds until the process exits,
 * which limits the lattice to LGF_NOALLOC_MAX_SITES = 2^20 sites (32^4); larger lattices get
 * LGF_ERR_UNSUPPORTED_SIZE (text from lgf_noalloc_last_error) and must use a context.  Extents 2 <= N <= 64.
 *   links_dev : device, LGF_LAYOUT_AOS [V][4][3][3] complex (FP64: 16 bytes each, FP32: 8), read only
 *   delta_dev : device, [V][3][3] complex, written; may be NULL (F and theta only)
 *   F_theta   : two doubles (F, theta), device or pinned host memory, written by a copy on the stream
 *   cuda_stream: a cudaStream_t passed as void*, may be NULL; the device that owns the buffers must be current.
 * Asynchronous: everything is enqueued on the stream, nothing is synchronised.  Calls cudaGetSymbolAddress once per
 * device; calls no cudaMalloc / cudaFree or any allocating routine.  All calls on one GPU SHARE the scratch array:
 * each call clears what must start at zero, but two calls that overlap on the GPU (different streams or host
 * threads) race -- serialise them.  Buffers are the caller's. */
#define LGF_NOALLOC_MAX_SITES 1048576
#define LGF_NOALLOC_SCRATCH_BYTES 131584
int lgf_measure_noalloc(int Nx, int Ny, int Nz, int Nt, int precision, const void *links_dev, void *delta_dev,
                        double *F_theta, void *cuda_stream);
/* Text of the last error of lgf_measure_noalloc in this process.  Never NULL. */
const char *lgf_noalloc_last_error(void);

/* Text of the last error of this context (or of lgf_create when ctx == NULL). Never NULL. */
const char *lgf_last_error(const lgf_ctx *ctx);

/* Free the context (host memory, events).  Caller buffers are never freed.  NULL is a no-op. */
int lgf_destroy(lgf_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* LGF_H */
