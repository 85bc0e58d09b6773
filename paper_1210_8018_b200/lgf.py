"""ctypes binding of liblgf.so (include/lgf.h).  Same names as the C ABI; argument marshalling
only -- every step of the gauge-fixing iteration runs in the CUDA kernels behind the library.

Low level: ``lib()`` returns the loaded CDLL with typed prototypes (``lgf_create`` ...).
Convenience: ``GaugeFixer`` owns a torch device workspace + stream and forwards to the ABI.
There is no CPU fallback: a missing or unloadable ``liblgf.so`` raises ``LgfError``.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# LGF_LIB_PATH: another build of the same library (same-run A/B of tuning macros); default: the in-tree build
LIB_PATH = os.environ.get("LGF_LIB_PATH") or os.path.join(_HERE, "liblgf.so")

OK = 0
ERR_INVALID_ARG, ERR_UNSUPPORTED_SIZE, ERR_NOT_BOUND, ERR_NOT_LOADED = -1, -2, -3, -4
ERR_WORKSPACE_TOO_SMALL, ERR_CUDA, ERR_NOT_CONVERGED, ERR_NUMERIC = -5, -6, -7, -8
PREC_FP64, PREC_FP32 = 0, 1
LAYOUT_AOS, LAYOUT_AOS12 = 0, 1
OPT_RECON, OPT_FFT_BATCH, OPT_MAX_ITER, OPT_CHECK_INTERVAL, OPT_FFT_PATH, OPT_PROFILE, OPT_FUSION, OPT_L2_PERSIST = 1, 2, 3, 4, 5, 6, 7, 8
OPT_GMAP, OPT_ACCUM_G, OPT_GRAPH, OPT_ZBLOCK, OPT_ZT_PIPE, OPT_FFT_PASSES = 9, 10, 11, 12, 13, 14
OPT_SHARD_WORLD, OPT_SHARD_RANK, OPT_TMARCH, OPT_LINK_TILE, OPT_LINK_STREAM = 15, 16, 17, 18, 19
(SHARD_MEASURE, SHARD_RESET, SHARD_XY_FWD, SHARD_PACK, SHARD_ZT, SHARD_UNPACK, SHARD_XY_INV_G, SHARD_LINK,
 SHARD_FINISH) = range(9)
REGION_CTRL, REGION_XSEND, REGION_XRECV, REGION_G, REGION_LINKS = range(5)
GMAP_FIRST_ORDER, GMAP_EXP = 0, 1
FIELD_DELTA, FIELD_W, FIELD_G = 0, 1, 2
STAGE_MEASURE, STAGE_FOURIER, STAGE_UPDATE = 0, 1, 2
KERNEL_NAMES = ["measure", "fft_xy_fwd", "fft_zt", "fft_xy_inv", "update", "fft_generic", "layout", "fft_xy_inv_g",
                "update_measure", "fft_xy_inv_gacc", "measure_acc", "apply_g"]

#: every symbol include/lgf.h declares
SYMBOLS = [
    "lgf_create", "lgf_set_option", "lgf_workspace_bytes", "lgf_bind", "lgf_load_links", "lgf_get_links",
    "lgf_measure", "lgf_iterate", "lgf_fix", "lgf_stage", "lgf_get_field", "lgf_set_field", "lgf_history",
    "lgf_kernel_time", "lgf_launch_count", "lgf_reset_counters", "lgf_uses_tiled_fft", "lgf_uses_gbuf", "lgf_zblock", "lgf_sync_links", "lgf_last_error",
    "lgf_destroy", "lgf_debug_dfma_rate", "lgf_shard_step", "lgf_shard_region", "lgf_shard_info", "lgf_shard_result",
    "lgf_measure_noalloc", "lgf_noalloc_last_error",
]


class LgfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"liblgf error {code}: {msg}")
        self.code = code


class lgf_result(ctypes.Structure):
    _fields_ = [("iterations", ctypes.c_int64), ("F", ctypes.c_double), ("theta", ctypes.c_double),
                ("converged", ctypes.c_int)]


_lib = None


def lib():
    """Load liblgf.so (no GPU needed to load it) and type its prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise LgfError(ERR_CUDA, f"{LIB_PATH} is missing: build it with `python -m paper_1210_8018_b200.build` "
                                 "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, i, i64, d = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double
    dp = ctypes.POINTER(ctypes.c_double)
    rp = ctypes.POINTER(lgf_result)
    L.lgf_create.argtypes = [i, i, i, i, i, ctypes.POINTER(vp)]
    L.lgf_set_option.argtypes = [vp, i, i64]
    L.lgf_workspace_bytes.argtypes = [vp]
    L.lgf_workspace_bytes.restype = ctypes.c_size_t
    L.lgf_bind.argtypes = [vp, vp, ctypes.c_size_t, vp]
    L.lgf_load_links.argtypes = [vp, vp, i, i]
    L.lgf_get_links.argtypes = [vp, vp, i, i]
    L.lgf_measure.argtypes = [vp, dp, dp]
    L.lgf_iterate.argtypes = [vp, d, i64, rp]
    L.lgf_fix.argtypes = [vp, d, d, rp]
    L.lgf_stage.argtypes = [vp, i, d]
    L.lgf_get_field.argtypes = [vp, i, d, vp, i]
    L.lgf_set_field.argtypes = [vp, i, vp, i]
    L.lgf_history.argtypes = [vp, dp, dp, i, ctypes.POINTER(i)]
    L.lgf_kernel_time.argtypes = [vp, i, dp, ctypes.POINTER(i64)]
    L.lgf_launch_count.argtypes = [vp]
    L.lgf_launch_count.restype = i64
    L.lgf_reset_counters.argtypes = [vp]
    L.lgf_uses_tiled_fft.argtypes = [vp]
    L.lgf_uses_gbuf.argtypes = [vp]
    L.lgf_zblock.argtypes = [vp]
    L.lgf_sync_links.argtypes = [vp]
    L.lgf_last_error.argtypes = [vp]
    L.lgf_last_error.restype = ctypes.c_char_p
    L.lgf_destroy.argtypes = [vp]
    L.lgf_debug_dfma_rate.argtypes = [vp, dp]
    L.lgf_shard_step.argtypes = [vp, i, d, d]
    L.lgf_shard_region.argtypes = [vp, i, ctypes.POINTER(ctypes.c_size_t), ctypes.POINTER(ctypes.c_size_t)]
    L.lgf_shard_info.argtypes = [vp, ctypes.POINTER(i64), i]
    L.lgf_shard_result.argtypes = [vp, rp]
    L.lgf_measure_noalloc.argtypes = [i, i, i, i, i, vp, vp, vp, vp]
    L.lgf_noalloc_last_error.argtypes = []
    L.lgf_noalloc_last_error.restype = ctypes.c_char_p
    _lib = L
    return L


def debug_dfma_rate(stream=None):
    """Measured FP64 FMA rate of the current device in DFMA/s (lgf_debug_dfma_rate)."""
    out = ctypes.c_double()
    rc = lib().lgf_debug_dfma_rate(stream, ctypes.byref(out))
    if rc:
        raise LgfError(rc, "lgf_debug_dfma_rate failed")
    return out.value


NOALLOC_MAX_SITES = 1 << 20


def measure_noalloc(N, links, delta, F_theta, stream=None):
    """lgf_measure_noalloc: Delta, F, theta of `links` (torch complex tensor on the GPU, [V,4,3,3]) into the
    caller's `delta` ([V,3,3], same dtype, or None) and `F_theta` (two float64, on the GPU or pinned host memory),
    enqueued on `stream` (a torch stream; default: the current one).  Allocates nothing; at most 2^20 sites.
    Marshalling only."""
    import torch

    N = _dims(N)
    prec = {torch.complex128: PREC_FP64, torch.complex64: PREC_FP32}[links.dtype]
    assert links.is_cuda and links.is_contiguous()
    assert delta is None or (delta.is_cuda and delta.is_contiguous() and delta.dtype == links.dtype)
    assert F_theta.dtype == torch.float64 and F_theta.numel() == 2 and F_theta.is_contiguous()
    with torch.cuda.device(links.device):
        st = stream if stream is not None else torch.cuda.current_stream(links.device)
        rc = lib().lgf_measure_noalloc(*N, prec, links.data_ptr(), delta.data_ptr() if delta is not None else None,
                                       F_theta.data_ptr(), st.cuda_stream)
    if rc:
        raise LgfError(rc, lib().lgf_noalloc_last_error().decode())


def _dims(N):
    N = (N,) * 4 if isinstance(N, int) else tuple(int(n) for n in N)
    assert len(N) == 4
    return N


class GaugeFixer:
    """One lattice on one GPU.  Thin wrapper: allocates the workspace with torch, binds it,
    and forwards every call to the C ABI.  Host arrays are numpy, complex128 (FP64 contexts)
    or complex64 (FP32 contexts), links [V,4,3,3], site fields [V,3,3]; device arrays are
    torch complex tensors of the same shapes."""

    def __init__(self, N, precision="fp64", recon=18, fft_batch=4, fft_path=0, device="cuda:0",
                 stream=None, max_iter=None, check_interval=None, profile=False, fusion=None, l2_persist=None, gmap=None,
                 accum_g=None, graph=None, zblock=None, zt_pipe=None, fft_passes=None, shard=None, tmarch=None, link_tile=None, link_stream=None):
        import torch

        self.torch = torch
        self.N = _dims(N)
        self.V = self.N[0] * self.N[1] * self.N[2] * self.N[3]
        if shard is not None:                   # (world, rank): this object holds one t-slab of the lattice N
            self.V //= int(shard[0])            # sites of the interchange arrays: the rank's own time slices
        self.prec = {"fp64": PREC_FP64, "fp32": PREC_FP32}[precision]
        self.np_dtype = np.complex128 if self.prec == PREC_FP64 else np.complex64
        self.torch_dtype = torch.complex128 if self.prec == PREC_FP64 else torch.complex64
        self.L = lib()
        self.ctx = ctypes.c_void_p()
        rc = self.L.lgf_create(*self.N, self.prec, ctypes.byref(self.ctx))
        if rc:
            raise LgfError(rc, self.L.lgf_last_error(None).decode())
        self.set_option(OPT_RECON, recon)
        self.set_option(OPT_FFT_BATCH, fft_batch)
        self.set_option(OPT_FFT_PATH, fft_path)
        if fusion is not None:
            self.set_option(OPT_FUSION, fusion)
        if l2_persist is not None:
            self.set_option(OPT_L2_PERSIST, l2_persist)
        if gmap is not None:
            self.set_option(OPT_GMAP, gmap)
        if accum_g is not None:
            self.set_option(OPT_ACCUM_G, accum_g)
        if graph is not None:
            self.set_option(OPT_GRAPH, graph)
        if zblock is not None:
            self.set_option(OPT_ZBLOCK, zblock)
        if zt_pipe is not None:
            self.set_option(OPT_ZT_PIPE, zt_pipe)
        if fft_passes is not None:
            self.set_option(OPT_FFT_PASSES, fft_passes)
        if tmarch is not None:
            self.set_option(OPT_TMARCH, tmarch)
        if link_tile is not None:
            self.set_option(OPT_LINK_TILE, link_tile)
        if link_stream is not None:
            self.set_option(OPT_LINK_STREAM, link_stream)
        if shard is not None:
            self.set_option(OPT_SHARD_WORLD, shard[0])
            self.set_option(OPT_SHARD_RANK, shard[1])
        if max_iter is not None:
            self.set_option(OPT_MAX_ITER, max_iter)
        if check_interval is not None:
            self.set_option(OPT_CHECK_INTERVAL, check_interval)
        if profile:
            self.set_option(OPT_PROFILE, 1)
        if not torch.cuda.is_available():
            raise LgfError(ERR_CUDA, "no CUDA device: liblgf has no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        nbytes = self.L.lgf_workspace_bytes(self.ctx)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        torch.cuda.synchronize(self.device)
        self._ck(self.L.lgf_bind(self.ctx, ptr, nbytes, self.stream.cuda_stream))

    # -- plumbing
    def _ck(self, rc, allow=()):
        if rc and rc not in allow:
            raise LgfError(rc, self.L.lgf_last_error(self.ctx).decode())
        return rc

    def close(self):
        if getattr(self, "ctx", None) is not None and self.ctx:
            self.L.lgf_destroy(self.ctx)
            self.ctx = ctypes.c_void_p()
            self.workspace = None       # hand the device memory back to torch

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _src(self, a, per_site):
        """(pointer, is_device, keepalive) for a numpy or torch array of V*per_site complex numbers."""
        torch = self.torch
        if isinstance(a, torch.Tensor):
            assert a.dtype == self.torch_dtype and a.is_contiguous() and a.numel() == self.V * per_site
            if a.is_cuda:
                # order the library's stream after whatever produced/consumes this tensor
                self.stream.wait_stream(torch.cuda.current_stream(self.device))
                return a.data_ptr(), 1, a
            return a.data_ptr(), 0, a
        assert isinstance(a, np.ndarray) and a.dtype == self.np_dtype and a.flags.c_contiguous
        assert a.size == self.V * per_site
        return a.ctypes.data, 0, a

    # -- the C ABI, same names
    def set_option(self, key, value):
        self._ck(self.L.lgf_set_option(self.ctx, key, int(value)))

    def workspace_bytes(self):
        return self.L.lgf_workspace_bytes(self.ctx)

    def load_links(self, U):
        """U: [V,4,3,3] (LAYOUT_AOS) or [V,4,2,3] (LAYOUT_AOS12: rows 0, 1), host or device."""
        rows2 = tuple(U.shape[-2:]) == (2, 3)
        p, dev, keep = self._src(U, 24 if rows2 else 36)
        self._ck(self.L.lgf_load_links(self.ctx, p, dev, LAYOUT_AOS12 if rows2 else LAYOUT_AOS))
        if dev:
            self.stream.synchronize()

    def get_links(self, out=None, device=False, rows=3):
        """rows = 3: [V,4,3,3] (LAYOUT_AOS); rows = 2: [V,4,2,3] (LAYOUT_AOS12)."""
        if out is None:
            out = (self.torch.empty((self.V, 4, rows, 3), dtype=self.torch_dtype, device=self.device) if device
                   else np.empty((self.V, 4, rows, 3), dtype=self.np_dtype))
        rows2 = tuple(out.shape[-2:]) == (2, 3)
        p, dev, keep = self._src(out, 24 if rows2 else 36)
        self._ck(self.L.lgf_get_links(self.ctx, p, dev, LAYOUT_AOS12 if rows2 else LAYOUT_AOS))
        return out

    def measure(self):
        F, th = ctypes.c_double(), ctypes.c_double()
        self._ck(self.L.lgf_measure(self.ctx, ctypes.byref(F), ctypes.byref(th)))
        return F.value, th.value

    def iterate(self, alpha, n, sync=True):
        if not sync:
            self._ck(self.L.lgf_iterate(self.ctx, float(alpha), int(n), None))
            return None
        r = lgf_result()
        self._ck(self.L.lgf_iterate(self.ctx, float(alpha), int(n), ctypes.byref(r)))
        return r

    def fix(self, alpha=0.08, eps=1e-15, allow_not_converged=False):
        r = lgf_result()
        self._ck(self.L.lgf_fix(self.ctx, float(alpha), float(eps), ctypes.byref(r)),
                 allow=(ERR_NOT_CONVERGED,) if allow_not_converged else ())
        return r

    def stage(self, stage, alpha=0.08):
        self._ck(self.L.lgf_stage(self.ctx, stage, float(alpha)))

    def get_field(self, which, alpha=0.08, device=False):
        out = (self.torch.empty((self.V, 3, 3), dtype=self.torch_dtype, device=self.device) if device
               else np.empty((self.V, 3, 3), dtype=self.np_dtype))
        p, dev, keep = self._src(out, 9)
        self._ck(self.L.lgf_get_field(self.ctx, which, float(alpha), p, dev))
        return out

    def set_field(self, which, a):
        p, dev, keep = self._src(a, 9)
        self._ck(self.L.lgf_set_field(self.ctx, which, p, dev))

    def history(self, cap=4096):
        F = np.empty(cap, dtype=np.float64)
        th = np.empty(cap, dtype=np.float64)
        n = ctypes.c_int()
        dp = ctypes.POINTER(ctypes.c_double)
        self._ck(self.L.lgf_history(self.ctx, F.ctypes.data_as(dp), th.ctypes.data_as(dp), cap, ctypes.byref(n)))
        return np.stack([F[: n.value], th[: n.value]], axis=1)

    def kernel_times(self):
        """{kind: (total ms, launches)} since the last reset (needs profile=True for the ms)."""
        out = {}
        for k, name in enumerate(KERNEL_NAMES):
            ms, cnt = ctypes.c_double(), ctypes.c_int64()
            self._ck(self.L.lgf_kernel_time(self.ctx, k, ctypes.byref(ms), ctypes.byref(cnt)))
            out[name] = (ms.value, cnt.value)
        return out

    def launch_count(self):
        return self.L.lgf_launch_count(self.ctx)

    def reset_counters(self):
        self._ck(self.L.lgf_reset_counters(self.ctx))

    def uses_tiled_fft(self):
        return bool(self.L.lgf_uses_tiled_fft(self.ctx))

    def uses_gbuf(self):
        return bool(self.L.lgf_uses_gbuf(self.ctx))

    def zblock(self):
        return int(self.L.lgf_zblock(self.ctx))

    # -- one lattice sharded over several GPUs (LGF_OPT_SHARD_WORLD): the steps and the exchanged regions
    def shard_step(self, step, alpha=0.0, eps=-1.0):
        self._ck(self.L.lgf_shard_step(self.ctx, int(step), float(alpha), float(eps)))

    def shard_region(self, region, dtype):
        """A torch view (1D, `dtype`) of an exchanged region of the workspace (include/lgf.h, LGF_REGION_*)."""
        off, nb = ctypes.c_size_t(), ctypes.c_size_t()
        self._ck(self.L.lgf_shard_region(self.ctx, int(region), ctypes.byref(off), ctypes.byref(nb)))
        base = (self.workspace.data_ptr() + 255) // 256 * 256 - self.workspace.data_ptr()
        return self.workspace[base + off.value: base + off.value + nb.value].view(dtype)

    def shard_info(self):
        a = (ctypes.c_int64 * 8)()
        self._ck(self.L.lgf_shard_info(self.ctx, a, 8))
        keys = ("stored_sites", "slice_sites", "own_slices", "ne", "elem_bytes", "world", "rank", "sites")
        return dict(zip(keys, [int(x) for x in a]))

    def shard_result(self):
        r = lgf_result()
        self._ck(self.L.lgf_shard_result(self.ctx, ctypes.byref(r)))
        return r

    def sync_links(self):
        self._ck(self.L.lgf_sync_links(self.ctx))

    def synchronize(self):
        self.stream.synchronize()
