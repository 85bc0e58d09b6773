"""A stream of independent lattices through ONE GPU with the transfers overlapped.

Gauge fixing is applied to ensembles of configurations (the paper's runs: sets of 32^4 lattices at several beta,
PAPER.md:171).  Through the C ABI one configuration costs  lgf_load_links (host -> device)  +  lgf_fix  +
lgf_get_links (device -> host), and at 32^4 the two PCIe transfers (403 MB each way with 12-real links) take as
long as the 50 iterations between them.  `EnsembleFixer` keeps `slots` contexts, each with its own CUDA stream and
workspace, and drives each from its own host thread (the ctypes calls release the interpreter lock): while one
slot computes, another uploads its next lattice and a third downloads its result, so upload, kernels and download
of different lattices overlap (full-duplex PCIe plus the SMs).  Marshalling only: every step still runs in the
kernels behind liblgf.so.  Host arrays should be pinned (page-locked), otherwise the copies are staged by the
driver and do not overlap.
"""
import threading

from . import lgf


class EnsembleFixer:
    def __init__(self, N, slots=3, device="cuda:0", **opts):
        """opts: keyword arguments of lgf.GaugeFixer (precision, recon, ...)."""
        self.fixers = [lgf.GaugeFixer(N, device=device, **opts) for _ in range(int(slots))]

    def run(self, inputs, outputs, alpha=0.08, eps=1e-15, iterations=None):
        """inputs[k] -> outputs[k] for every k: load, fix to theta <= eps (or exactly `iterations` iterations when
        given), get.  inputs / outputs: sequences of host arrays in an interchange layout of the context.  Returns
        the list of lgf_result, in input order.  Lattice k is handled by slot k mod slots."""
        n = len(inputs)
        results = [None] * n
        errors = []

        def work(slot):
            gf = self.fixers[slot]
            try:
                for k in range(slot, n, len(self.fixers)):
                    gf.load_links(inputs[k])
                    results[k] = gf.iterate(alpha, iterations) if iterations is not None else gf.fix(alpha, eps, allow_not_converged=True)
                    gf.get_links(out=outputs[k])
            except Exception as e:          # noqa: BLE001 -- re-raised in the caller's thread below
                errors.append(e)

        threads = [threading.Thread(target=work, args=(s,)) for s in range(min(len(self.fixers), n))]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        if errors:
            raise errors[0]
        return results

    def close(self):
        for f in self.fixers:
            f.close()
