"""bench.py -- throughput of the gauge-fixing hot path (arXiv 1210.8018, Algorithm 1) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 32^4] [--impl ours|reference]

A step is one execution of the loop body of Algorithm 1 (FFT filter of Delta, g build, link
update, measure) on one lattice.  Default workload: BASELINE.json configs[2], the headline
32^4 FP64 lattice with 12-real links.  Metric: site-iterations/s = V * steps / time.
With N > 1 (torchrun) every rank fixes its own lattice (replicas, no data-path collective:
DESIGN.md section 9), `value` is the sum over ranks / max time over ranks.

One JSON line on stdout (rank 0).  `value` is device-resident; `e2e` goes through the C ABI
with pinned HOST buffers every step: lgf_load_links (H2D), lgf_iterate(1), lgf_get_links (D2H);
`e2e.fix` is the time to solution the same way (load, lgf_fix to theta <= eps, get the links).
`--impl reference` times the CPU oracle (oracle/) instead, as it stands, on the host cores.
`--gpus N` without a torchrun environment starts the N ranks itself (re-exec under
`python -m torch.distributed.run`, rendezvous on 127.0.0.1).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "gauge-fix site-iterations/s"
UNIT = "site-iterations/s"
ALPHA = 0.08

# workload name -> (extents, sigma, seed offset, precision, recon)   (BASELINE.json `configs`)
WORKLOADS = {
    "8^4": ((8,) * 4, 0.3, 8, "fp64", 18),
    "16^4": ((16,) * 4, 0.5, 16, "fp64", 18),
    "32^4": ((32,) * 4, 0.5, 32, "fp64", 12),
    "48^4": ((48,) * 4, 0.5, 48, "fp32", 18),
    "64^4": ((64,) * 4, 0.6, 64, "fp64", 18),
}


def workload_label(args, prec, recon, seed, sigma):
    """config.workload: the same string in both arms (--impl ours / reference time the same named workload)."""
    return (f"{args.workload} periodic SU(3), {prec}, {recon}-real links, {args.fft_batch} FFT fields, "
            f"alpha={ALPHA}, gen seed {seed}, sigma={sigma}"
            + (", ACCUM_G (fixed links + accumulated G, link rewrite inside the window)" if args.accum_g else "")
            + (", g = exp((alpha/2) w)" if args.gmap else ""))


def algorithmic_bytes(recon, nfields, real_bytes, tiled, fusion, gbuf, accum=0):
    """Bytes per site each kernel must move once:
    L = link bytes per site, W = field bytes per site, Gb = bytes of rows 0, 1 of g per site."""
    L = 4 * recon * real_bytes
    W = nfields * 2 * real_bytes
    Gb = 12 * real_bytes
    per = {}
    if accum:
        # LGF_OPT_ACCUM_G: links read once, never written; G read by the link kernel, read + written by the last pass
        return {"measure_acc": L + Gb + W, "fft_xy_fwd": 2 * W, "fft_zt": 2 * W, "fft_xy_inv_gacc": W + 2 * Gb}
    if fusion:
        per["update_measure"] = (Gb if gbuf else W) + 2 * L + W
    else:
        per.update({"measure": L + W, "update": W + 2 * L})
    if tiled:
        per.update({"fft_xy_fwd": 2 * W, "fft_zt": 2 * W})
        per.update({"fft_xy_inv_g": W + Gb} if gbuf else {"fft_xy_inv": 2 * W})
    else:
        per["fft_generic"] = 2 * W       # per launch (8 launches per iteration)
    return per


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def mark(self):
        return time.time()

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.1] or [r for (_, r) in self.rows]
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(workload_key, kernel):
    """(DRAM bytes per launch of `kernel`, where the number comes from) out of the committed ncu summaries
    (profiles/*_traffic.csv; the latest file that has the row wins), or (None, None).  The bench run itself
    cannot measure DRAM traffic (that takes ncu, and a number taken under a profiler is never a bench value),
    so `traffic_source` names the csv file, the capture the row belongs to and the commit that added the file."""
    import csv
    import glob

    best, src = None, None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv"))):
        with open(path) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload_key and row["kernel"] == kernel:
                    best = int(row["dram_read_bytes"]) + int(row["dram_write_bytes"])
                    src = {"file": os.path.relpath(path, ROOT), "capture": row.get("capture") or os.path.basename(path).split("_")[0]}
    if src:
        try:
            src["commit"] = subprocess.run(["git", "-C", ROOT, "log", "-1", "--format=%h", "--", src["file"]],
                                           capture_output=True, text=True, timeout=10).stdout.strip() or None
        except (OSError, subprocess.SubprocessError):
            src["commit"] = None
        if not src["commit"]:           # no git history here (GPU boxes): the "commit:" line of the .md beside the csv
            try:
                for line in open(os.path.join(ROOT, src["file"][:-4] + ".md")):
                    if line.startswith("commit:"):
                        src["commit"] = line.split()[1]
            except OSError:
                pass
    return best, src


def time_oracle(N, sigma, seed, iters):
    """The oracle as it stands, single thread: site-iterations/s over `iters` iterations."""
    import gen
    import oracle

    U = gen.gen_links(N, sigma, seed)
    oracle.measure(N, U, want_delta=False)          # page everything in
    t = time.perf_counter()
    oracle.iterate(N, U, ALPHA, iters)
    dt = time.perf_counter() - t
    V = N[0] * N[1] * N[2] * N[3]
    return V * iters / dt, dt


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, one bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import gen

    N, sigma, soff, prec, recon = WORKLOADS[args.workload]
    # a step = one oracle iteration (about 3 s at 32^4 on one core) on the lattice the line names.  Lattices
    # above 32^4 (tens of seconds per oracle iteration) are bounded to their 32^4 corner of the same generator,
    # and config.workload then says so.
    Ns = tuple(min(n, 32) for n in N)
    seed = gen.BASE_SEED + soff
    import oracle

    U = gen.gen_links(Ns, sigma, seed)
    Vs = Ns[0] * Ns[1] * Ns[2] * Ns[3]
    for _ in range(args.warmup):
        oracle.iterate(Ns, U, ALPHA, 1)
    t = time.perf_counter()
    for _ in range(args.steps):
        oracle.iterate(Ns, U, ALPHA, 1)
    dt = time.perf_counter() - t
    val = Vs * args.steps / dt
    sample = f"{args.steps} single-thread oracle iterations on {'x'.join(map(str, Ns))} (same generator, sigma={sigma}, seed {seed})"
    ran = "x".join(map(str, Ns))
    workload = workload_label(args, prec, args.recon or recon, seed, sigma)
    if Ns != tuple(N):
        workload += f" [oracle timed on its {ran} corner: bounded sample]"
    sample += "; the oracle as it stands: FP64, 18-real AoS links, one FFT per element of Delta (9), one thread"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload, "lattice": list(Ns), "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; liblgf has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator log (stderr) shows the ranks that joined
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_1210_8018_b200 import build as lgf_build
    from paper_1210_8018_b200 import lgf

    if rank == 0:
        lgf_build.build()
    if world > 1:
        dist.barrier()
    import gen

    N, sigma, soff, prec, recon = WORKLOADS[args.workload]
    if args.recon:
        recon = args.recon
    V = N[0] * N[1] * N[2] * N[3]
    from paper_1210_8018_b200 import replicas

    seed = replicas.replica_seed(gen.BASE_SEED + soff, rank)   # every rank its own lattice (replicas)
    U = gen.gen_links(N, sigma, seed)
    cdt = np.complex128 if prec == "fp64" else np.complex64
    tdt = torch.complex128 if prec == "fp64" else torch.complex64
    U = U.astype(cdt, copy=False)
    host = torch.empty((V, 4, 3, 3), dtype=tdt).pin_memory()
    host.copy_(torch.from_numpy(U))
    dev = host.to(f"cuda:{local}")
    torch.cuda.synchronize()

    gf = lgf.GaugeFixer(N, precision=prec, recon=recon, fft_batch=args.fft_batch, fft_path=args.fft_path,
                        fusion=args.fusion, l2_persist=args.l2_persist, accum_g=args.accum_g, gmap=args.gmap, graph=args.graph,
                        zblock=args.zblock, zt_pipe=args.zt_pipe, link_tile=args.link_tile, link_stream=args.link_stream, tmarch=args.tmarch, device=f"cuda:{local}")
    K, W = args.steps, args.warmup
    stream = gf.stream

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed_iterations(profile):
        """W untimed + K timed iterations from the freshly loaded links; returns (ms, launches)."""
        gf.set_option(lgf.OPT_PROFILE, 0)
        gf.load_links(dev)
        gf.iterate(ALPHA, W)
        gf.load_links(dev)                      # timed window = iterations 1..K of Algorithm 1
        gf.set_option(lgf.OPT_PROFILE, 1 if profile else 0)
        gf.reset_counters()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        with torch.cuda.stream(stream):
            e0.record(stream)
            gf.iterate(ALPHA, K, sync=False)
            gf.sync_links()                     # ACCUM_G: the one link rewrite belongs to the window; else a no-op
            e1.record(stream)
        barrier()
        return e0.elapsed_time(e1), gf.launch_count()

    # ---- device-resident timing (the headline `value`)
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
        time.sleep(0.15)
    t0 = time.time()
    ms, launches = timed_iterations(profile=False)
    t1 = time.time()
    r_end = gf.iterate(ALPHA, 0)

    # ---- time to solution: Algorithm 1 from the loaded links to theta <= eps (context, not the metric)
    fix_eps = 1e-15 if prec == "fp64" else 1e-12
    gf.load_links(dev)
    torch.cuda.synchronize()
    tf = time.perf_counter()
    r_fix = gf.fix(ALPHA, fix_eps, allow_not_converged=True)
    fix_ms = 1e3 * (time.perf_counter() - tf)

    # ---- the same window with every launch bracketed by CUDA events on the library's stream
    ms_prof, _ = timed_iterations(profile=True)
    ktimes = gf.kernel_times()
    gf.set_option(lgf.OPT_PROFILE, 0)

    # ---- end to end through the C ABI with pinned host buffers, copies inside the timed region
    e2e_steps = K
    # 12-real contexts take the 12-real exchange format (LGF_LAYOUT_AOS12: rows 0, 1), two thirds of the bytes
    per_link = 6 if recon == 12 else 9
    if per_link == 6:
        host12 = torch.empty((V, 4, 2, 3), dtype=tdt).pin_memory()
        host12.copy_(host[:, :, :2, :])
        host = host12
    host_out = torch.empty_like(host).pin_memory()
    gf.load_links(host.numpy())
    gf.get_links(out=host_out.numpy())
    barrier()
    te = time.perf_counter()
    for _ in range(e2e_steps):
        gf.load_links(host.numpy())             # H2D of the step's input (4 x per_link complex per site)
        gf.iterate(ALPHA, 1)                    # one iteration + D2H of (iterations, F, theta)
        gf.get_links(out=host_out.numpy())      # D2H of the step's result: the transformed links, same layout
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - te
    # time to solution through the same calls: load -> lgf_fix -> get (how the library is used)
    barrier()
    tf2 = time.perf_counter()
    gf.load_links(host.numpy())
    r_fix2 = gf.fix(ALPHA, fix_eps, allow_not_converged=True)
    gf.get_links(out=host_out.numpy())
    torch.cuda.synchronize()
    fix_e2e_s = time.perf_counter() - tf2
    # the same steps for a STREAM of lattices (ensembles are the use case): three contexts, streams and host
    # threads, so that the upload of one lattice, the kernels of another and the download of a third overlap (ensemble.py)
    pipe_s = pipe_fix_s = None
    if args.pipeline and world == 1 and V <= 48 ** 4:          # 64^4 would pin another 30 GB of host memory for the three slots
        try:
            from paper_1210_8018_b200 import ensemble

            ens = ensemble.EnsembleFixer(N, slots=3, precision=prec, recon=recon, fft_batch=args.fft_batch, device=f"cuda:{local}")
            pouts = [torch.empty_like(host).pin_memory() for _ in range(3)]
            ens.run([host.numpy()] * 3, [p.numpy() for p in pouts], ALPHA, iterations=1)          # warm-up
            torch.cuda.synchronize()
            tp = time.perf_counter()
            ens.run([host.numpy()] * e2e_steps, [pouts[k % 3].numpy() for k in range(e2e_steps)], ALPHA, iterations=1)
            torch.cuda.synchronize()
            pipe_s = time.perf_counter() - tp
            # and the time to solution for a stream of lattices: load, lgf_fix, get per lattice, three in flight
            nfix = 12
            tq = time.perf_counter()
            rq = ens.run([host.numpy()] * nfix, [pouts[k % 3].numpy() for k in range(nfix)], ALPHA, fix_eps)
            torch.cuda.synchronize()
            pipe_fix_s = (time.perf_counter() - tq, nfix, int(rq[0].iterations))
            ens.close()
            del pouts
        except Exception as e:                                  # noqa: BLE001
            pipe_s = None
            sys.stderr.write(f"bench.py: pipelined e2e leg skipped: {e}\n")
    clocks = sampler.stop(t0, t1) if sampler else None
    try:
        dfma_rate = lgf.debug_dfma_rate(stream.cuda_stream)     # measured FP64 FMA rate: the "alu" denominator
    except Exception:                                           # noqa: BLE001
        dfma_rate = None

    (ms_all, e2e_all, fix_e2e_all), _ = replicas.reduce_timing([ms, e2e_s, fix_e2e_s], V * K, device=f"cuda:{local}")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    real_bytes = 8 if prec == "fp64" else 4
    tiled = gf.uses_tiled_fft()
    per = algorithmic_bytes(recon, args.fft_batch, real_bytes, tiled, args.fusion, gf.uses_gbuf(), args.accum_g)
    peak, peak_src = peaks()
    kern = {k: {"ms_total": v[0], "launches": v[1], "us_per_launch": 1e3 * v[0] / v[1]}
            for k, v in ktimes.items() if v[1] and k in per}
    for k in kern:
        kern[k]["bytes_per_site"] = per[k]
        kern[k]["GBps"] = per[k] * V / (kern[k]["us_per_launch"] * 1e-6) / 1e9
        kern[k]["share"] = kern[k]["ms_total"] / sum(v[0] for kk, v in ktimes.items() if kk in per)
    dom = max(kern, key=lambda k: kern[k]["ms_total"])
    # the analytic minimum of the three-kernel design, 3 L + 8 W bytes per site and
    # iteration (1664 for 12-real FP64, 2240 for 18-real FP64, 1120 for 18-real FP32 with 4 packed
    # fields), is the yardstick whatever this build actually moves; `moved` is what it must move
    Lb, Wb = 4 * recon * real_bytes, args.fft_batch * 2 * real_bytes
    iter_bytes = 3 * Lb + 8 * Wb
    moved_bytes = sum(per[k] * (8 if k == "fft_generic" else 1) for k in per)
    value = world * V * K / (ms_all * 1e-3)
    e2e_val = world * V * e2e_steps / e2e_all
    h2d = V * 4 * per_link * 2 * real_bytes

    # ---- side-by-side reference only (never on the product path): cuFFT through torch.fft on the same
    # number of fields, forward + inverse 4D transforms, against the three hand-written passes
    # ---- the ACCUM_G variant of the same workload, same run, same window (context: faster, moves fewer bytes)
    variants = None
    if world == 1 and not args.accum_g and tiled and gf.uses_gbuf() and args.variants:
        try:
            ga = lgf.GaugeFixer(N, precision=prec, recon=recon, fft_batch=args.fft_batch, accum_g=1, gmap=args.gmap,
                                graph=args.graph, device=f"cuda:{local}")
            ga.load_links(dev)
            ga.iterate(ALPHA, W)
            ga.load_links(dev)
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            with torch.cuda.stream(ga.stream):
                a0.record(ga.stream)
                ga.iterate(ALPHA, K, sync=False)
                ga.sync_links()                 # the one link rewrite belongs to the window
                a1.record(ga.stream)
            torch.cuda.synchronize()
            ams = a0.elapsed_time(a1)
            variants = {"accum_g": {"ms_per_step": ams / K, "value": V * K / (ams * 1e-3), "unit": UNIT,
                                    "bytes_per_site_this_build": 4 * recon * real_bytes + 6 * Wb + 3 * 12 * real_bytes,
                                    "what": "LGF_OPT_ACCUM_G = 1: fixed links + accumulated transformation, link rewrite "
                                            "inside the window (bench.py --accum-g 1 makes it the timed path)"}}
            ga.close()
        except Exception as e:                  # noqa: BLE001
            variants = {"accum_g": {"unavailable": str(e).splitlines()[0][:160]}}

    # ---- two independent lattices iterating at the same time on this GPU (one context and stream each): the link kernel of
    # one overlaps the FFT passes of the other.  Context for ensembles; the headline stays one lattice.
    if world == 1 and args.variants and not args.accum_g:
        try:
            import threading

            pair = [gf, lgf.GaugeFixer(N, precision=prec, recon=recon, fft_batch=args.fft_batch, gmap=args.gmap,
                                       graph=args.graph, stream=torch.cuda.Stream(device=f"cuda:{local}"), device=f"cuda:{local}")]
            for g in pair:
                g.load_links(dev)
                g.iterate(ALPHA, W)
            torch.cuda.synchronize()
            e0 = torch.cuda.Event(enable_timing=True)
            ends = [torch.cuda.Event(enable_timing=True) for _ in pair]
            e0.record(pair[0].stream)
            pair[1].stream.wait_event(e0)

            def run(g, e):
                g.iterate(ALPHA, K, sync=False)
                e.record(g.stream)

            ths = [threading.Thread(target=run, args=(g, e)) for g, e in zip(pair, ends)]
            for t in ths:
                t.start()
            for t in ths:
                t.join()
            torch.cuda.synchronize()
            tms = max(e0.elapsed_time(e) for e in ends)
            variants = dict(variants or {})
            variants["two_lattices"] = {"ms_per_round": tms / K, "value": 2 * V * K / (tms * 1e-3), "unit": UNIT,
                                        "what": "aggregate of two independent lattices of this workload iterating concurrently "
                                                "(two contexts, two streams): one round = one iteration of each"}
            pair[1].close()
        except Exception as e:                  # noqa: BLE001
            variants = dict(variants or {})
            variants["two_lattices"] = {"unavailable": str(e).splitlines()[0][:160]}

    fft_ref = None
    if tiled and args.cufft_reference:
        try:
            del dev
            f = torch.randn((args.fft_batch, N[3], N[2], N[1], N[0]), dtype=tdt, device=f"cuda:{local}")
            for _ in range(3):
                f = torch.fft.ifftn(torch.fft.fftn(f, dim=(1, 2, 3, 4)), dim=(1, 2, 3, 4))
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            c0.record()
            for _ in range(10):
                f = torch.fft.ifftn(torch.fft.fftn(f, dim=(1, 2, 3, 4)), dim=(1, 2, 3, 4))
            c1.record()
            torch.cuda.synchronize()
            ours = sum(kern[k]["us_per_launch"] for k in kern if k.startswith("fft_")) * 1e-3
            fft_ref = {"cufft_fwd_inv_ms": c0.elapsed_time(c1) / 10, "ours_3_passes_ms": ours,
                       "note": "cuFFT (torch.fft.fftn + ifftn, no mask, no g build) vs this build's passes (mask, 1/V and g build included)"}
            del f
        except RuntimeError as e:       # out of memory on the largest lattices: the reference is optional
            fft_ref = {"unavailable": str(e).splitlines()[0][:120]}

    # ---- CPU baseline: the oracle as it stands on a bounded sample of the same workload
    cpu = None
    if not args.no_cpu_baseline:
        Ns = N if V <= 32 ** 4 else tuple(min(n, 32) for n in N)
        iters = {True: 3}.get(Ns[0] >= 32, 20 if Ns[0] >= 16 else 200)
        v, dt = time_oracle(Ns, sigma, gen.BASE_SEED + soff, iters)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{iters} oracle iterations on {'x'.join(map(str, Ns))} ({dt:.1f} s, single thread, "
                         f"{os.cpu_count()} cores on the box)"}

    traffic, traffic_src = ncu_traffic(f"{args.workload}-{prec}-recon{recon}-fields{args.fft_batch}", dom)
    # FP64 instructions (DFMA + DMUL + DADD) per site of the link kernels, counted in the SASS of this build up to the block
    # reduction (cuobjdump -sass, profiles/r02_sass.md): 12-real 1182 + 289 + 176, 18-real 1038 + 241 + 188 (ACCUM_G 18-real: sum form)
    fp64_per_site = {"update_measure": 1647 if recon == 12 else 1467, "measure_acc": 1647 if recon == 12 else 1316}
    alu = None
    if dfma_rate:
        nominal = 148 * 64 * 1.965e9
        alu = {"peak": dfma_rate, "unit": "FP64 instructions/s (DFMA rate measured by lgf_debug_dfma_rate in this run)",
               "nominal": nominal, "nominal_what": "148 SMs x 64 DFMA/clk x 1.965 GHz", "kernels": {}}
        for k in kern:
            if k in fp64_per_site and prec == "fp64":
                a = fp64_per_site[k] * V / (kern[k]["us_per_launch"] * 1e-6)
                alu["kernels"][k] = {"fp64_instructions_per_site": fp64_per_site[k], "achieved": a, "frac": a / dfma_rate}
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_all / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if prec == "fp64" else "f32", "data": "synthetic",
        "config": {"workload": workload_label(args, prec, recon, gen.BASE_SEED + soff, sigma),
                   "lattice": list(N), "zblock": gf.zblock(), "zt_pipe": args.zt_pipe, "link_tile": args.link_tile, "link_stream": args.link_stream,
                   "fft": "tiled register FFT, 3 passes" if tiled else "generic per-axis transform, 8 passes",
                   "l2": "working set (links + fields) exceeds the 126 MB L2" if V >= 32 ** 4 else
                         "working set fits in L2; latency/L2-bound by design (DESIGN.md section 6)",
                   "parallelism": "replicas" if world > 1 else "single GPU",
                   "final": {"iterations": int(r_end.iterations), "F": r_end.F, "theta": r_end.theta},
                   "fix": {"eps": fix_eps, "iterations": int(r_fix.iterations), "converged": int(r_fix.converged),
                           "F": r_fix.F, "theta": r_fix.theta, "wall_ms": fix_ms}},
        "clocks": clocks,
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": h2d + 32,
                "ms_per_step": 1e3 * e2e_all / e2e_steps,
                "what": "every step: lgf_load_links(pinned host, " + ("12-real rows 0-1 layout" if per_link == 6 else "18-real layout")
                        + ") + lgf_iterate(1) with its (iterations, F, theta) readback + lgf_get_links(pinned host, same layout)",
                "pipelined": (None if pipe_s is None else
                              {"what": "the same step (load, one iteration, get) for a stream of lattices through ensemble.EnsembleFixer: 3 contexts, "
                                       "streams and host threads on this GPU, transfers of different lattices overlapped",
                               "value": V * e2e_steps / pipe_s, "unit": UNIT, "ms_per_step": 1e3 * pipe_s / e2e_steps}),
                "fix": {"what": "time to solution through the same calls: lgf_load_links(host) + lgf_fix(alpha, eps) + lgf_get_links(host)",
                        "eps": fix_eps, "iterations": int(r_fix2.iterations), "converged": int(r_fix2.converged),
                        "ms": 1e3 * fix_e2e_all, "value": world * V * int(r_fix2.iterations) / fix_e2e_all, "unit": UNIT,
                        "h2d_bytes": h2d, "d2h_bytes": h2d + 32,
                        "pipelined": (None if pipe_fix_s is None else
                                      {"what": f"{pipe_fix_s[1]} lattices through ensemble.EnsembleFixer (3 in flight), each load + lgf_fix + get",
                                       "ms_per_lattice": 1e3 * pipe_fix_s[0] / pipe_fix_s[1], "iterations": pipe_fix_s[2],
                                       "value": V * pipe_fix_s[2] * pipe_fix_s[1] / pipe_fix_s[0], "unit": UNIT})}},
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": kern[dom]["GBps"], "peak": peak, "unit": "GB/s",
                     "frac": kern[dom]["GBps"] / peak,
                     "traffic": traffic, "traffic_source": traffic_src,
                     "algorithmic_bytes": per[dom] * V, "peak_source": peak_src,
                     "bytes_per_site": per[dom],
                     # the whole iteration against the bytes THIS build must move (sum of the kernels' algorithmic
                     # bytes); the three-kernel yardstick of SURVEY 8(d) (3 L + 8 W) is kept as a separate, named field
                     "iteration": {"bytes_per_site": moved_bytes, "GBps": moved_bytes * V * K / (ms_all * 1e-3) / 1e9,
                                   "frac": moved_bytes * V * K / (ms_all * 1e-3) / 1e9 / peak,
                                   "survey_yardstick": {"bytes_per_site": iter_bytes,
                                                        "GBps_equivalent": iter_bytes * V * K / (ms_all * 1e-3) / 1e9,
                                                        "frac_equivalent": iter_bytes * V * K / (ms_all * 1e-3) / 1e9 / peak,
                                                        "what": "SURVEY 8(d) row for this config (3 L + 8 W bytes per site): what a "
                                                                "three-kernel design would have to move in the same time; not real traffic"},
                                   "ms_profiled": ms_prof / K},
                     # second roofline, plain FP64 arithmetic: FP64 instructions per site of the link kernels (SASS
                     # count, profiles/) against the DFMA rate measured in this run by lgf_debug_dfma_rate
                     "alu": alu,
                     "kernels": kern},
        "cpu_baseline": cpu,
        "fft_reference": fft_ref,
        "variants": variants,
    }
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_launch_selftest(args):
    """--launch-selftest: what `--gpus N` starts, without the lattice work: every rank joins the process
    group (nccl on GPUs, gloo when there is none: the CPU test of the launcher), the step-time reduction
    of DESIGN.md section 9 runs once, rank 0 prints how many ranks took part."""
    import torch
    import torch.distributed as dist

    from paper_1210_8018_b200 import replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cuda = torch.cuda.is_available() and torch.cuda.device_count() >= world
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if cuda:
            torch.cuda.set_device(local)
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")
    times, units = replicas.reduce_timing([1.0 + rank], 1.0, device=f"cuda:{local}" if cuda else "cpu")
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"launch_selftest": True, "n_gpus": world, "ranks_counted": int(units), "max_ms": times[0],
                          "backend": "nccl" if cuda else "gloo"}), flush=True)


def spawn_ranks(n):
    """`python bench.py --gpus N` outside torchrun: start the N ranks (one per GPU) by re-executing this
    command line under `python -m torch.distributed.run` with a rendezvous on 127.0.0.1, pass their
    output through and return their exit code.  Rank 0 prints the JSON line."""
    import socket

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="32^4", choices=sorted(WORKLOADS))
    ap.add_argument("--recon", type=int, default=0, choices=[0, 12, 18])
    ap.add_argument("--fft-batch", type=int, default=4, choices=[4, 9])
    ap.add_argument("--fft-path", type=int, default=0, choices=[0, 1])
    ap.add_argument("--fusion", type=int, default=1, choices=[0, 1])
    ap.add_argument("--l2-persist", type=int, default=0, choices=[0, 1])
    ap.add_argument("--accum-g", type=int, default=0, choices=[0, 1],
                    help="LGF_OPT_ACCUM_G: fixed links + accumulated transformation (the link rewrite at the end of the window is timed)")
    ap.add_argument("--variants", type=int, default=1, choices=[0, 1], help="also time the ACCUM_G variant (N = 1)")
    ap.add_argument("--graph", type=int, default=1, choices=[0, 1], help="LGF_OPT_GRAPH (default on)")
    ap.add_argument("--gmap", type=int, default=0, choices=[0, 1], help="LGF_OPT_GMAP: 1 = exact exponential")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cufft-reference", type=int, default=1, choices=[0, 1])
    ap.add_argument("--pipeline", type=int, default=1, choices=[0, 1], help="also time the e2e step for a stream of lattices (ensemble.py)")
    ap.add_argument("--zblock", type=int, default=None, help="LGF_OPT_ZBLOCK (default: chosen from the L2 size)")
    ap.add_argument("--link-tile", type=int, default=None, help="LGF_OPT_LINK_TILE: 1 = site kernel, 128 / 256 / 512 = threads per 4D tile")
    ap.add_argument("--link-stream", type=int, default=None, choices=[0, 1], help="LGF_OPT_LINK_STREAM: 1 = TMA-fed persistent link kernel")
    ap.add_argument("--tmarch", type=int, default=None, help="LGF_OPT_TMARCH")
    ap.add_argument("--zt-pipe", type=int, default=None, choices=[0, 1], help="LGF_OPT_ZT_PIPE")
    ap.add_argument("--launch-selftest", action="store_true", help="start the ranks, reduce one timing, print the rank count")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args.gpus))
    if "WORLD_SIZE" in os.environ and int(os.environ["WORLD_SIZE"]) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ['WORLD_SIZE']}")
    if args.launch_selftest:
        run_launch_selftest(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
