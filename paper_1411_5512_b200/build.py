"""Build libea_b200.so (the product: hand-written sm_100a kernels + the C ABI of include/ea.h) in-tree.

`python -m paper_1411_5512_b200.build` or `build()` from `__graft_entry__.build()`.  nvcc cross-compiles
without a GPU.  The library links the CUDA runtime statically: no torch, no Python.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libea_b200.so")
SOURCES = ["ea_api.cu", "ea_sweep.cu", "ea_sweep_resident.cu", "ea_sweep_small.cu", "ea_setup.cu", "ea_observables.cu",
           "ea_c4_vectors.cu", "ea_fold.cu", "ea_pipes.cu"]
HEADERS = ["ea_device.cuh", "ea_sweep_common.cuh", "ea_internal.h", os.path.join("..", "..", "include", "ea.h")]
ARCH_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMPILE_FLAGS = ARCH_FLAGS + ["-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]
LINK_FLAGS = ARCH_FLAGS + ["-shared", "-cudart", "static"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src: str, obj: str, verbose: bool):
    cmd = [_nvcc()] + COMPILE_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
    return src, subprocess.run(cmd, capture_output=True, text=True)


def build(force: bool = False, verbose: bool = False) -> str:
    """One nvcc -c per source file, in parallel (objects are cached under build/ by source mtime; `force` recompiles
    all of them), then one link."""
    if not force and not needs_build():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    hdr_t = max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)
    hdr_t = max(hdr_t, os.path.getmtime(os.path.abspath(__file__)))
    jobs, objs = [], []
    for f in SOURCES:
        src, obj = os.path.join(CSRC, f), os.path.join(objdir, f[:-3] + ".o")
        objs.append(obj)
        stale = not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_t)
        if stale or verbose or force:
            jobs.append((src, obj))
    with ThreadPoolExecutor(max_workers=max(1, min(len(jobs), os.cpu_count() or 1))) as ex:
        for src, res in ex.map(lambda j: _compile(j[0], j[1], verbose), jobs):
            if res.returncode != 0:
                sys.stderr.write(res.stdout + res.stderr)
                raise RuntimeError("nvcc failed compiling %s" % src)
            if verbose:
                sys.stderr.write(res.stdout + res.stderr)
    tmp = LIB + ".tmp.%d" % os.getpid()
    res = subprocess.run([_nvcc()] + LINK_FLAGS + ["-o", tmp] + objs, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking libea_b200.so")
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--incremental" not in sys.argv, verbose="-v" in sys.argv))
