"""Build libcsf.so (hand-written sm_100a kernels + C ABI) in-tree with nvcc.

The shared object lands next to this file (paper_2410_02754_b200/libcsf.so) so that it travels to the GPU
box with the repo snapshot. nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcsf.so")
SOURCES = ["csf_api.cu", "csf_tables.cpp", "csf_column_p.cu", "csf_colws_p.cu"]
HEADERS = ["csf_kernels.cuh", "csf_column.cuh", "csf_colws.cuh", "csf_subspace.cuh", "csf_dense.cuh", "csf_column_launch.h", "csf_tables.h", os.path.join("..", "..", "include", "csf.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--use_fast_math=false",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def _run(cmd):
    res = subprocess.run(cmd, capture_output=True, text=True)
    return res.returncode, res.stdout + res.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    """nvcc -c every translation unit in parallel (one per FE order for the column kernel), then link libcsf.so."""
    if not force and not _stale():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    cflags = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]
    cflags += os.environ.get("CSF_NVCC_EXTRA", "").split()         # e.g. -DCSF_WIDE_AUXW=2 for a tuning build
    jobs = [(os.path.join(CSRC, "csf_api.cu"), os.path.join(objdir, "csf_api.o"), []),
            (os.path.join(CSRC, "csf_tables.cpp"), os.path.join(objdir, "csf_tables.o"), [])]
    jobs += [(os.path.join(CSRC, "csf_column_p.cu"), os.path.join(objdir, f"csf_column_p{p}.o"), [f"-DCSF_P={p}"]) for p in range(1, 8)]
    jobs += [(os.path.join(CSRC, "csf_column_p.cu"), os.path.join(objdir, f"csf_column_wide_p{p}.o"), [f"-DCSF_P={p}", "-DCSF_WIDE=1"]) for p in (4, 5)]
    # the wide order-5 FP64 kernel with two gather warps (fused projector gather of csf_filter's half-block path)
    jobs += [(os.path.join(CSRC, "csf_column_p.cu"), os.path.join(objdir, "csf_column_wide_p5_g.o"), ["-DCSF_P=5", "-DCSF_WIDE=1", "-DCSF_GATHERW=2"])]
    jobs += [(os.path.join(CSRC, "csf_colws_p.cu"), os.path.join(objdir, f"csf_colws_p{p}.o"), [f"-DCSF_P={p}"]) for p in (4, 5)]
    with ThreadPoolExecutor(max_workers=min(12, os.cpu_count() or 2)) as ex:
        results = list(ex.map(lambda j: _run(["nvcc"] + cflags + j[2] + ["-c", j[0], "-o", j[1]]), jobs))
    log = "".join(out for _, out in results)
    if verbose or any(rc != 0 for rc, _ in results):
        sys.stderr.write(log)
    if any(rc != 0 for rc, _ in results):
        raise RuntimeError("nvcc failed building libcsf.so")
    rc, out = _run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + [j[1] for j in jobs] + ["-ldl"])
    if rc != 0:
        sys.stderr.write(out)
        raise RuntimeError("nvcc failed linking libcsf.so")
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
        f.write(log + out)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
