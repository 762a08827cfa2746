"""Build libnoit.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnoit.so")
SOURCES = ["noit_api.cu", "noit_features.cu", "noit_resolve.cu", "noit_resolve_staged.cu",
           "noit_quadtree.cu", "noit_reproject.cu"]
# no -use_fast_math anywhere: IEEE division / sqrt are part of the bit-exact classes
COMMON = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
          "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-I", CSRC]
PER_FILE = {"noit_reproject.cu": ["-fmad=false"], "noit_quadtree.cu": ["-fmad=false"]}


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "noit.h"),
                                                               os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


DEBUG_LIB = os.path.join(HERE, "libnoit_debug.so")     # staged kernel with -DNOIT_DEBUG_BOUNDS
DEBUG_SRC = "noit_resolve_staged.cu"


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every CUDA translation unit and link libnoit.so -- and libnoit_debug.so, the same
    objects with the staged resolve kernel compiled with -DNOIT_DEBUG_BOUNDS (own bounds checks;
    tests/test_steps_gpu.py runs the parity cases through it).  Returns libnoit.so's path."""
    if not force and not _stale() and os.path.exists(DEBUG_LIB):
        return LIB
    nvcc = _nvcc()
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    procs = []
    jobs = [(src, src.replace(".cu", ".o"), []) for src in SOURCES]
    jobs.append((DEBUG_SRC, DEBUG_SRC.replace(".cu", "_debug.o"), ["-DNOIT_DEBUG_BOUNDS"]))
    for src, oname, extra in jobs:
        obj = os.path.join(objdir, oname)
        cmd = [nvcc, *COMMON, *PER_FILE.get(src, []), *extra, *(["-Xptxas", "-v"] if verbose else []),
               "-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((src, obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)))
    objs = []
    for src, obj, pr in procs:
        out, _ = pr.communicate()
        if verbose or pr.returncode != 0:
            sys.stderr.write(out.decode(errors="replace"))
        if pr.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(obj)
    link = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"]
    release = objs[:-1]
    debug = [objs[-1] if o.endswith(DEBUG_SRC.replace(".cu", ".o")) else o for o in release]
    subprocess.check_call([*link, "-o", LIB, *release])
    subprocess.check_call([*link, "-o", DEBUG_LIB, *debug])
    return LIB


def build_variant(name: str, defines: list, verbose: bool = False) -> str:
    """A/B build: libnoit_<name>.so = the release objects with the staged resolve kernel recompiled
    with the given -D flags (NOIT_X_WARPS, NOIT_X_CTAS, NOIT_X_STAGE, NOIT_X_WSMEM; see
    noit_resolve_staged.cu).  Select it with NOIT_LIBRARY=<path> (binding.lib) and time it with
    `python bench.py --config cfgK`: how the occupancy experiments of profiles/r02_resolve.md were run."""
    build()
    nvcc = _nvcc()
    objdir = os.path.join(HERE, "build")
    obj = os.path.join(objdir, f"noit_resolve_staged_{name}.o")
    cmd = [nvcc, *COMMON, *defines, *(["-Xptxas", "-v"] if verbose else []), "-c",
           os.path.join(CSRC, DEBUG_SRC), "-o", obj]
    out = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)
    if verbose or out.returncode != 0:
        sys.stderr.write(out.stdout.decode(errors="replace"))
    if out.returncode != 0:
        raise RuntimeError("nvcc failed on the variant")
    objs = [obj if src == DEBUG_SRC else os.path.join(objdir, src.replace(".cu", ".o")) for src in SOURCES]
    lib = os.path.join(HERE, f"libnoit_{name}.so")
    subprocess.check_call([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart", "-o", lib, *objs])
    return lib


if __name__ == "__main__":
    if "--variant" in sys.argv:
        i = sys.argv.index("--variant")
        print(build_variant(sys.argv[i + 1], [a for a in sys.argv[i + 2:] if a.startswith("-D")], verbose="-v" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
