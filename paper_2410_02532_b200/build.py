"""Build libopo.so (hand-written sm_100a kernels + the C ABI of include/opo.h) in-tree with nvcc.

    python -m paper_2410_02532_b200.build [--force]

nvcc cross-compiles without a GPU.  The result, paper_2410_02532_b200/libopo.so, is git-ignored but
travels to the GPU box with the working tree.
"""
from __future__ import annotations

import os
import re
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libopo.so")
PLAIN_SOURCES = ["opo_api.cu", "opo_dispatch.cu", "opo_pointwise.cu", "opo_selftest.cu"]
# (type, suffix, log2 N): one object per size-specialised instance of opo_inst.cu
INSTANCES = [("float", "f32", l) for l in range(4, 15)] + [("double", "f64", l) for l in range(4, 14)]
# wide engine (a cluster of 4 F CTAs per instance): the sizes whose plan is 4 . 16 . r . r'
WIDE_INSTANCES = [("float", "f32", l) for l in range(12, 15)] + [("double", "f64", l) for l in range(12, 14)]
LARGE_INSTANCES = [("float", "f32", l) for l in range(15, 19)] + [("double", "f64", l) for l in range(14, 19)]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _newest_source_mtime() -> float:
    paths = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if os.path.isfile(os.path.join(CSRC, f))]
    paths.append(os.path.join(os.path.dirname(HERE), "include", "opo.h"))
    return max(os.path.getmtime(p) for p in paths)


_INCLUDE = re.compile(r'^\s*#\s*include\s*"([^"]+)"', re.M)
_DEPS = {}


def _deps_mtime(path: str) -> float:
    """Newest modification time of a source and of every file it includes with "..." (recursively)."""
    path = os.path.normpath(path)
    if path in _DEPS:
        return _DEPS[path]
    _DEPS[path] = m = os.path.getmtime(path)
    with open(path) as f:
        for inc in _INCLUDE.findall(f.read()):
            cand = os.path.normpath(os.path.join(os.path.dirname(path), inc))
            if os.path.exists(cand):
                m = max(m, _deps_mtime(cand))
    _DEPS[path] = m
    return m


def _jobs(only=None):
    jobs = [(src, src.replace(".cu", ".o"), []) for src in PLAIN_SOURCES]
    for typ, suf, l in INSTANCES:
        if only and f"{suf}:{l}" not in only:
            continue
        jobs.append(("opo_inst.cu", f"opo_inst_{suf}_L{l}.o", [f"-DOPO_T={typ}", f"-DOPO_SUFFIX={suf}", f"-DOPO_L={l}"]))
        # the N/2 - L - N/2 instantiation of the resident kernel, in an object of its own
        jobs.append(("opo_inst.cu", f"opo_inst_nln_{suf}_L{l}.o", [f"-DOPO_T={typ}", f"-DOPO_SUFFIX={suf}", f"-DOPO_L={l}", "-DOPO_NLN"]))
        # the dk = 0 instantiation (no stage phases in RK4), likewise
        jobs.append(("opo_inst.cu", f"opo_inst_dk0_{suf}_L{l}.o", [f"-DOPO_T={typ}", f"-DOPO_SUFFIX={suf}", f"-DOPO_L={l}", "-DOPO_NLN", "-DOPO_DK0"]))
        # the solo engine (one CTA per instance, fields in shared + tensor memory): general and dk = 0 instantiations
        jobs.append(("opo_inst_solo.cu", f"opo_inst_solo_{suf}_L{l}.o", [f"-DOPO_T={typ}", f"-DOPO_SUFFIX={suf}", f"-DOPO_L={l}"]))
        jobs.append(("opo_inst_solo.cu", f"opo_inst_solo_dk0_{suf}_L{l}.o", [f"-DOPO_T={typ}", f"-DOPO_SUFFIX={suf}", f"-DOPO_L={l}", "-DOPO_DK0"]))
        # ... and its pump-train instantiation (slices in, exit fields out at the round-trip crossings inside the launch)
        jobs.append(("opo_inst_solo.cu", f"opo_inst_solo_train_{suf}_L{l}.o", [f"-DOPO_T={typ}", f"-DOPO_SUFFIX={suf}", f"-DOPO_L={l}", "-DOPO_TRAIN"]))
    for typ, suf, l in WIDE_INSTANCES:
        if only and f"{suf}:{l}" not in only:
            continue
        jobs.append(("opo_inst_wide.cu", f"opo_inst_wide_{suf}_L{l}.o", [f"-DOPO_T={typ}", f"-DOPO_SUFFIX={suf}", f"-DOPO_L={l}"]))
        jobs.append(("opo_inst_wide.cu", f"opo_inst_wide_dk0_{suf}_L{l}.o", [f"-DOPO_T={typ}", f"-DOPO_SUFFIX={suf}", f"-DOPO_L={l}", "-DOPO_DK0"]))
    for typ, suf, l in LARGE_INSTANCES:
        if only and f"{suf}:{l}" not in only:
            continue
        jobs.append(("opo_inst_large.cu", f"opo_inst_large_{suf}_L{l}.o", [f"-DOPO_T={typ}", f"-DOPO_SUFFIX={suf}", f"-DOPO_L={l}"]))
    return jobs


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every CUDA source for sm_100a and link libopo.so.  OPO_BUILD_ONLY="f32:14,f64:10"
    (development only) restricts the size-specialised instances; sizes left out report
    OPO_ERR_UNSUPPORTED at opo_create.  OPO_EXTRA_NVCC_FLAGS (diagnostic builds, e.g. -DOPO_LARGE_TIMING) is
    appended to every compile; use it with --force and rebuild without it afterwards."""
    only = os.environ.get("OPO_BUILD_ONLY")
    only = set(only.split(",")) if only else None
    if not force and not only and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source_mtime():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    _DEPS.clear()

    def compile_one(job) -> str:
        src, objname, defs = job
        obj = os.path.join(OBJ, objname)
        # an object is stale when its source or a header it includes is newer
        if not force and os.path.exists(obj) and os.path.getmtime(obj) >= _deps_mtime(os.path.join(CSRC, src)):
            return obj
        cmd = [nvcc, *NVCC_FLAGS, *os.environ.get("OPO_EXTRA_NVCC_FLAGS", "").split(), *defs, "-c", os.path.join(CSRC, src), "-o", obj]
        res = subprocess.run(cmd, capture_output=True, text=True)
        with open(obj + ".log", "w") as f:
            f.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src} {defs}:\n{res.stdout}\n{res.stderr}")
        if verbose:
            print(res.stderr)
        return obj

    jobs = _jobs(only)
    for src in sorted({j[0] for j in jobs}):        # fill the dependency cache before the threads start: _deps_mtime is not
        _deps_mtime(os.path.join(CSRC, src))        # re-entrant (a half-computed entry would hide a changed header)
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        objs = list(ex.map(compile_one, jobs))
    cmd = [nvcc, "-shared", "-o", LIB, *objs, "-cudart", "static", "-ldl"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError(f"link failed:\n{res.stdout}\n{res.stderr}")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
