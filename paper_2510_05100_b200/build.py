"""Build librex_trex.so (the C-ABI CUDA library) in-tree for sm_100a.  `python -m paper_2510_05100_b200.build [--force]`."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librex_trex.so")
# (source, object stem, extra defines); the g g -> t t~ + gluons kernels are compiled once per (N, precision mode)
UNITS = [("trex_ttng_tu.cu", "trex_ttng_n%d_m%d" % (n, m), ["-DTREX_TU_N=%d" % n, "-DTREX_TU_MODE=%d" % m])
         for n in (5, 4, 3, 2) for m in (0, 1, 2)] + \
        [("trex_table_tu.cu", "trex_table_n%d_m%d" % (n, m), ["-DTREX_TU_N=%d" % n, "-DTREX_TU_MODE=%d" % m])
         for n in (5, 4, 3) for m in (0, 1, 2)] + [("trex_api.cu", "trex_api", []), ("trex_qq2_tu.cu", "trex_qq2", []), ("rex_bucket.cu", "rex_bucket", []),
                                                 ("trex_probe.cu", "trex_probe", []), ("trex_xsec.cu", "trex_xsec", [])]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-Wno-deprecated-gpu-targets"]


# headers each source depends on (besides itself)
_KERNEL_HDRS = ["trex_math.cuh", "trex_ttng.cuh", "trex_proc.cuh", "trex_kernels.cuh", "trex_ctx.h", "../../include/rex_trex.h", "../../include/rex_trex_diag.h"]
DEPS = {
    "trex_ttng_tu.cu": _KERNEL_HDRS,
    "trex_table_tu.cu": _KERNEL_HDRS + ["trex_table.cuh", "trex_table4.cuh"],
    "trex_qq2_tu.cu": _KERNEL_HDRS + ["trex_qq2.cuh"],
    "trex_api.cu": _KERNEL_HDRS + ["trex_ctx.h", "trex_host.h", "trex_colour.h", "../../include/rex_trex.h"],
    "rex_bucket.cu": ["trex_ctx.h", "../../include/rex_trex.h"],
    "trex_probe.cu": ["trex_ctx.h", "../../include/rex_trex.h"],
    "trex_xsec.cu": ["trex_ctx.h", "../../include/rex_trex.h"],
}


def _src_mtime(src):
    return max(os.path.getmtime(os.path.join(CSRC, f)) for f in [src] + DEPS[src] + ["../build.py"])


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def build(force=False, verbose=False):
    stale = [u for u in UNITS
             if force or not os.path.exists(os.path.join(HERE, "build", u[1] + ".o"))
             or os.path.getmtime(os.path.join(HERE, "build", u[1] + ".o")) < _src_mtime(u[0])]
    if not stale and os.path.exists(LIB):
        return LIB
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    objs = [os.path.join(HERE, "build", stem + ".o") for _, stem, _ in UNITS]

    def compile_one(unit):
        src, stem, defs = unit
        obj = os.path.join(HERE, "build", stem + ".o")
        cmd = [nvcc()] + NVCC_FLAGS + defs + ["-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        with open(os.path.join(HERE, "build", stem + ".log"), "w") as fh:
            fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s" % (stem, r.stderr[-4000:]))
        if verbose:
            sys.stderr.write(r.stderr)

    if stale:
        with ThreadPoolExecutor(max(1, min(len(stale), os.cpu_count() or 1))) as ex:
            list(ex.map(compile_one, stale))
    subprocess.check_call([nvcc(), "-shared", "-o", LIB] + objs + ["-lcudart"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
