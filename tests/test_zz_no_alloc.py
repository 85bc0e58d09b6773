"""lgf_measure_noalloc (include/lgf.h, csrc/noalloc.cu): the one entry point that allocates nothing -- its scratch
memory is a static device array -- against the existing context path (lgf_create / lgf_bind / lgf_load_links /
lgf_measure / lgf_get_field) and the oracle, on calls in a row that share that array.

Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test.  Passes alone in a
fresh process and after the other tests: it keeps no state but the library's own static array, which every call
clears where it must."""
import ctypes

import numpy as np
import pytest

import gen
import oracle

# tolerances of tests/test_gpu_parity.py::test_measure_matches_oracle
TOL = {"fp64": dict(delta=1e-13, rel=1e-12), "fp32": dict(delta=2e-5, rel=1e-5)}


def close_F(F, Fref, rel):
    # F starts near 0 on a random gauge: relative to max(|F|, 1e-3), as test_measure_matches_oracle does
    return abs(F - Fref) <= rel * max(abs(Fref), 1e-3) + 1e-15


@pytest.fixture(scope="module")
def lgf(cuda_device):
    from paper_1210_8018_b200 import lgf as m

    m.lib()
    return m


def context_path(lgf, N, U, prec):
    gf = lgf.GaugeFixer(N, precision=prec, recon=18)
    gf.load_links(U)
    F, th = gf.measure()
    D = gf.get_field(lgf.FIELD_DELTA)
    gf.close()
    return F, th, D


@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_measure_noalloc_matches_the_context_path_on_calls_in_a_row(lgf, prec):
    """Three calls in a row on one stream, each on another lattice (the second smaller than the first, so stale
    partial sums of the first call lie behind the ones it uses; the third ends in a half-filled last CTA):
    Delta, F and theta equal the context path's within the tolerances of the parity tests, and the oracle's."""
    import torch

    cdt = np.complex128 if prec == "fp64" else np.complex64
    tol = TOL[prec]
    cases = [((16, 16, 16, 16), 0.5, 4101), ((8, 12, 6, 4), 0.3, 4102), ((6, 4, 12, 18), 0.5, 4103)]
    outs = []
    for N, sigma, seed in cases:                       # enqueue all three before looking at any result
        U = gen.gen_links(N, sigma, seed).astype(cdt)
        Ud = torch.from_numpy(U).cuda()
        Dd = torch.full((U.shape[0], 3, 3), float("nan"), dtype=Ud.dtype, device="cuda")
        ft = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
        lgf.measure_noalloc(N, Ud, Dd, ft)
        outs.append((N, U, Ud, Dd, ft))
    torch.cuda.synchronize()
    for N, U, Ud, Dd, ft in outs:
        F, th = (float(x) for x in ft.cpu())
        D = Dd.cpu().numpy()
        Fc, thc, Dc = context_path(lgf, N, U, prec)
        assert np.abs(D - Dc).max() <= tol["delta"], N
        assert close_F(F, Fc, tol["rel"]) and abs(th - thc) <= tol["rel"] * thc, (N, F, Fc, th, thc)
        Do, Fo, tho = oracle.measure(N, U.astype(np.complex128))
        assert np.abs(D.astype(np.complex128) - Do).max() <= tol["delta"], N
        assert close_F(F, Fo, tol["rel"]) and abs(th - tho) <= tol["rel"] * tho, (N, F, Fo, th, tho)


@pytest.mark.gpu
def test_measure_noalloc_repeats_bitwise_and_takes_the_largest_lattice(lgf):
    """The same input twice in a row gives bitwise the same numbers (the second call starts from the first call's
    leftovers), also without a Delta output and with the result in pinned host memory; 32^4 = LGF_NOALLOC_MAX_SITES is
    accepted and agrees with the context path."""
    import torch

    N = (32, 32, 32, 32)
    assert N[0] * N[1] * N[2] * N[3] == lgf.NOALLOC_MAX_SITES
    U = gen.gen_links(N, 0.5, gen.BASE_SEED + 32)
    Ud = torch.from_numpy(U).cuda()
    Dd = torch.empty((U.shape[0], 3, 3), dtype=Ud.dtype, device="cuda")
    ft1 = torch.zeros(2, dtype=torch.float64, device="cuda")
    ft2 = torch.zeros(2, dtype=torch.float64).pin_memory()
    lgf.measure_noalloc(N, Ud, Dd, ft1)
    D1 = Dd.clone()
    lgf.measure_noalloc(N, Ud, None, ft2)
    lgf.measure_noalloc(N, Ud, Dd, ft1)
    torch.cuda.synchronize()
    assert torch.equal(D1, Dd)
    assert ft1.cpu().tolist() == ft2.tolist()
    Fc, thc, Dc = context_path(lgf, N, U, "fp64")
    assert np.abs(Dd.cpu().numpy() - Dc).max() <= 1e-13
    assert close_F(ft2[0].item(), Fc, 1e-12) and abs(ft2[1].item() - thc) <= 1e-12 * thc


def test_measure_noalloc_rejects_what_it_cannot_hold():
    """Host-side validation, before any CUDA call: more sites than the static scratch array covers, bad extents,
    bad precision, NULL buffers -- each with a clear text."""
    from paper_1210_8018_b200 import build, lgf

    build.build()
    L = lgf.lib()
    dummy = ctypes.c_void_p(256)
    assert L.lgf_measure_noalloc(48, 48, 48, 48, lgf.PREC_FP32, dummy, None, dummy, None) == lgf.ERR_UNSUPPORTED_SIZE
    msg = L.lgf_noalloc_last_error().decode()
    assert "5308416 sites exceed LGF_NOALLOC_MAX_SITES = 1048576" in msg and "context" in msg
    assert L.lgf_measure_noalloc(32, 32, 32, 34, lgf.PREC_FP64, dummy, None, dummy, None) == lgf.ERR_UNSUPPORTED_SIZE
    assert L.lgf_measure_noalloc(8, 8, 8, 128, lgf.PREC_FP64, dummy, None, dummy, None) == lgf.ERR_UNSUPPORTED_SIZE
    assert L.lgf_measure_noalloc(8, 1, 8, 8, lgf.PREC_FP64, dummy, None, dummy, None) == lgf.ERR_UNSUPPORTED_SIZE
    assert L.lgf_measure_noalloc(8, 8, 8, 8, 5, dummy, None, dummy, None) == lgf.ERR_INVALID_ARG
    assert L.lgf_measure_noalloc(8, 8, 8, 8, lgf.PREC_FP64, None, None, dummy, None) == lgf.ERR_INVALID_ARG
    assert L.lgf_measure_noalloc(8, 8, 8, 8, lgf.PREC_FP64, dummy, None, None, None) == lgf.ERR_INVALID_ARG
    assert b"NULL" in L.lgf_noalloc_last_error()
