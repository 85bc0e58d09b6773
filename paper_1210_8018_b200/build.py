"""Build paper_1210_8018_b200/liblgf.so in-tree with nvcc for sm_100a.

    python -m paper_1210_8018_b200.build [--force]

nvcc cross-compiles without a GPU.  Objects go to paper_1210_8018_b200/build/ (git-ignored);
the shared library sits beside this file so that it travels to the GPU box with the repo.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liblgf.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
ZT_EXTENTS = [8, 12, 16, 24, 32, 48, 64]
# (source, extra flags, object name); fft_zt_inst.cu is compiled once per Nz (the (z,t) pass of the tiled FFT
# for that Nz and every Nt), so that the 7 x 7 extent pairs build in parallel
SOURCES = [(f, [], f.replace(".cu", ".o")) for f in
           ["lgf_api.cu", "kernels_site.cu", "kernels_fused.cu", "fft_generic.cu", "fft_tiled.cu", "microbench.cu", "noalloc.cu"]]
SOURCES += [("fft_zt_inst.cu", [f"-DLGF_ZT_NA={n}"], f"fft_zt_na{n}.o") for n in ZT_EXTENTS]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Wno-deprecated-gpu-targets", "-I", INCLUDE,
]


def _nvcc():
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.sep not in p or os.path.exists(p)):
            return p
    raise RuntimeError("nvcc not found")


def _deps_mtime():
    m = 0.0
    for d in (CSRC, INCLUDE):
        for f in os.listdir(d):
            m = max(m, os.path.getmtime(os.path.join(d, f)))
    return max(m, os.path.getmtime(os.path.abspath(__file__)))


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu of csrc/ for sm_100a and link liblgf.so.  Returns its path."""
    newest = _deps_mtime()
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()

    def compile_one(item):
        src, flags, objname = item
        obj = os.path.join(OBJ, objname)
        if not force and os.path.exists(obj) and os.path.getmtime(obj) >= newest:
            return obj
        extra = flags + os.environ.get("LGF_EXTRA_NVCC_FLAGS", "").split()    # tuning macros of csrc/*.cu for same-run A/B builds (-DLGF_FUSED_BWD_REV=1 ...)
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError(f"nvcc failed on {src} {' '.join(flags)}")
        return obj

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    subprocess.check_call([nvcc, "-shared", "-o", LIB] + objs + ["-lcudart"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
