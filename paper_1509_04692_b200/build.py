"""Build libhpmc.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo snapshot).

The library is several translation units (the C-ABI + cell-list kernels, and one per family of colour-pass kernels) that
are compiled in parallel and linked; no relocatable device code is needed, every kernel is self-contained.
"""
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "_obj")
LIB = os.path.join(HERE, "libhpmc.so")
UNITS = ["hpmc_api", "pass_colour", "pass_tile2d_disk", "pass_tile2d_pentagon", "pass_tile2d_polygon", "pass_warpcell_2d",
         "pass_warpcell_3d", "pass_warpcell_3d_nv", "pass_cluster2d", "pass_spec2d", "noalloc_count"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _newest_source() -> float:
    t = 0.0
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for f in os.listdir(root):
            t = max(t, os.path.getmtime(os.path.join(root, f)))
    return t


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)

    def compile_unit(u):
        cmd = [nvcc] + NVCC_FLAGS + ["-c", os.path.join(CSRC, u + ".cu"), "-o", os.path.join(OBJ, u + ".o")]
        return u, cmd, subprocess.run(cmd, capture_output=True, text=True)

    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_unit, UNITS))
    log = []
    for u, cmd, res in results:
        # the register / spill report, without the timing lines that change from build to build
        log.append(" ".join(cmd) + "\n" + "\n".join(l for l in res.stderr.splitlines() if "Compile time" not in l) + "\n")
        if verbose or res.returncode != 0:
            print(res.stdout)
            print(res.stderr)
        if res.returncode != 0:
            raise RuntimeError(f"nvcc failed compiling {u}.cu")
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "--shared", "-Xcompiler", "-fPIC", "-o", LIB] + \
           [os.path.join(OBJ, u + ".o") for u in UNITS]
    res = subprocess.run(link, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed linking libhpmc.so")
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
        f.write("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
