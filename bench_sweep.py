"""Variant sweep on 32^3 x n lattices: the shape of Fig. 1 of arXiv 1210.8018 (PAPER.md:140,
165-169, 183) on one B200.

    python bench_sweep.py [--nt 8 16 32 48 64] [--steps 20] [--out sweep.md]

Variants: single / double precision x 18 / 12 reals per link (the paper's sp/dp and 18/12-real
axes; its texture and ECC axes are Fermi board settings).  For every variant
and lattice it times `steps` iterations of Algorithm 1 with lgf_iterate (CUDA events on the
library's stream, 5 warm-up iterations) and prints a markdown table: ms per iteration,
site-iterations/s, and the GFlops the PAPER'S flop model would credit for that rate
(Table 1, plus V 5 (log2(nx ny) + log2(nz nt)) per 4D FFT, 9 forward and
9 inverse) -- the unit of the paper's 186 / 71 GFlops on a Tesla C2070
(PAPER.md:185).  This build executes fewer operations than that model counts (4 packed FFT fields,
rows-only link products), so the figure is a rate in the paper's currency, not an operation count.
Inputs are the seeded synthetic generator of DESIGN.md section 4 (sigma = 0.5).

    python bench_sweep.py --passes [--nt ...]

times the paper's third axis instead, the decomposition of the 4D FFT ("The best choice for our
4D problem is two 2D FFTs"), same run, same lattices, FP64 12-real and FP32 18-real: the fused
three-pass default (2D | 2D * mask * 2D | 2D), 2D + 2D as four passes (LGF_OPT_FFT_PASSES = 4, the paper's best),
4 x 1D as eight passes with the same register lines (= 8), and the generic per-axis O(N^2) transform
(LGF_OPT_FFT_PATH = 1).  3D + 1D is not built (it needs a cluster-wide DSMEM transpose).
Columns: ms per iteration and the time of the FFT passes alone (CUDA events around every launch).
"""
import argparse
import math
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def paper_flops_per_site(N, recon):
    """Flop count per site and iteration in the paper's model (Table 1 + FFT model)."""
    k2, k5, k6 = (841, 153, 1962) if recon == 12 else (505, 153, 1584)
    k4 = 2 * 9
    fft = 18 * 5 * (math.log2(N[0] * N[1]) + math.log2(N[2] * N[3]))
    return k2 + k4 + k5 + k6 + fft


def alpha_scan(alphas, sizes, gen, lgf):
    """Iterations of Algorithm 1 until theta <= 1e-15 as a function of the step alpha (eq. 1.2,
    PAPER.md:49; the paper fixes alpha = 0.08) for g = reunit(1 + (alpha/2) w) and for
    g = exp((alpha/2) w), on the synthetic N^4 lattices of DESIGN.md section 4."""
    lines = ["| lattice | alpha | g map | iterations | final F | final theta | converged |", "|---|---|---|---|---|---|---|"]
    for n in sizes:
        U = gen.gen_links(n, 0.5, gen.BASE_SEED + n)
        import torch
        Ud = torch.from_numpy(U).cuda()
        for gmap, name in ((0, "first order + reunit"), (1, "exp")):
            gf = lgf.GaugeFixer(n, recon=12, gmap=gmap, max_iter=400)
            for al in alphas:
                gf.load_links(Ud)
                try:
                    r = gf.fix(al, 1e-15, allow_not_converged=True)
                except lgf.LgfError as e:       # theta became NaN/Inf: the step is too long
                    lines.append(f"| {n}^4 | {al:.4f} | {name} | - | - | - | diverged ({e.code}) |")
                    continue
                lines.append(f"| {n}^4 | {al:.4f} | {name} | {r.iterations} | {r.F:.12f} | {r.theta:.3e} | {r.converged} |")
            gf.close()
        del Ud
    return "\n".join(lines)


def passes_sweep(nts, steps, gen, lgf):
    import numpy as np
    import torch

    structures = [("3 passes: 2D | 2D mask 2D | 2D (default)", dict()),
                  ("4 passes: 2D + 2D (the paper's best, P:119)", dict(fft_passes=4)),
                  ("8 passes: 4 x 1D, register lines", dict(fft_passes=8)),
                  ("8 passes: per-axis O(N^2) transform (generic path)", dict(fft_path=1))]
    lines = ["| lattice | precision | reals/link | FFT structure | FFT launches/iteration | ms/iteration | FFT passes alone, ms | site-iterations/s |",
             "|---|---|---|---|---|---|---|---|"]
    for nt in nts:
        N = (32, 32, 32, nt)
        V = 32 * 32 * 32 * nt
        U = gen.gen_links(N, 0.5, gen.BASE_SEED + 3200 + nt)
        for prec, recon in (("fp64", 12), ("fp32", 18)):
            Ud = torch.from_numpy(U.astype(np.complex64 if prec == "fp32" else np.complex128)).cuda()
            for name, opt in structures:
                try:
                    gf = lgf.GaugeFixer(N, precision=prec, recon=recon, **opt)
                except lgf.LgfError as e:
                    lines.append(f"| 32^3 x {nt} | {prec} | {recon} | {name} | - | not available ({e.code}) | - | - |")
                    continue
                gf.load_links(Ud)
                gf.iterate(0.08, 5)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                with torch.cuda.stream(gf.stream):
                    e0.record(gf.stream)
                    gf.iterate(0.08, steps, sync=False)
                    e1.record(gf.stream)
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1) / steps
                gf.set_option(lgf.OPT_PROFILE, 1)
                gf.reset_counters()
                gf.iterate(0.08, steps)
                kt = gf.kernel_times()
                fft_ms = sum(v[0] for k, v in kt.items() if k.startswith("fft_")) / steps
                nl = sum(v[1] for k, v in kt.items() if k.startswith("fft_")) // steps
                lines.append(f"| 32^3 x {nt} | {prec} | {recon} | {name} | {nl} | {ms:.4f} | {fft_ms:.4f} | {V / (ms * 1e-3):.3e} |")
                gf.close()
            del Ud
    return "\n".join(lines)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--nt", type=int, nargs="+", default=[8, 16, 32, 48, 64])
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--out", default=None)
    ap.add_argument("--alpha-scan", type=float, nargs="*", default=None,
                    help="instead of the timing sweep: iterations to theta <= 1e-15 for these alpha, both g maps")
    ap.add_argument("--scan-n", type=int, nargs="+", default=[16, 32])
    ap.add_argument("--passes", action="store_true", help="instead of the precision / storage sweep: the FFT pass-structure axis")
    args = ap.parse_args()
    import numpy as np
    import torch

    import gen
    from paper_1210_8018_b200 import lgf

    if args.alpha_scan is not None:
        text = alpha_scan(args.alpha_scan or [0.04, 0.05, 0.0625, 0.07, 0.08, 0.09, 0.10, 0.11, 0.12], args.scan_n, gen, lgf)
        print(text)
        if args.out:
            with open(args.out, "w") as f:
                f.write(text + "\n")
        return

    if args.passes:
        text = passes_sweep(args.nt, args.steps, gen, lgf)
        print(text)
        if args.out:
            with open(args.out, "w") as f:
                f.write(text + "\n")
        return

    lines = ["| lattice | precision | reals/link | FFT path | ms/iteration | site-iterations/s | paper-model GFlops |",
             "|---|---|---|---|---|---|---|"]
    for nt in args.nt:
        N = (32, 32, 32, nt)
        V = 32 * 32 * 32 * nt
        U = gen.gen_links(N, 0.5, gen.BASE_SEED + 3200 + nt)
        for prec in ("fp32", "fp64"):
            Ud = torch.from_numpy(U.astype(np.complex64 if prec == "fp32" else np.complex128)).cuda()
            for recon in (18, 12):
                gf = lgf.GaugeFixer(N, precision=prec, recon=recon)
                gf.load_links(Ud)
                gf.iterate(0.08, 5)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                with torch.cuda.stream(gf.stream):
                    e0.record(gf.stream)
                    gf.iterate(0.08, args.steps, sync=False)
                    e1.record(gf.stream)
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1) / args.steps
                rate = V / (ms * 1e-3)
                lines.append(f"| 32^3 x {nt} | {prec} | {recon} | {'tiled' if gf.uses_tiled_fft() else 'generic'} | {ms:.4f} | "
                             f"{rate:.3e} | {rate * paper_flops_per_site(N, recon) / 1e9:.0f} |")
                gf.close()
            del Ud
    text = "\n".join(lines)
    print(text)
    if args.out:
        with open(args.out, "w") as f:
            f.write(text + "\n")


if __name__ == "__main__":
    main()
