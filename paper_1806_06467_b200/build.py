"""Build libfresnel.so IN-TREE with nvcc for sm_100a (no JIT cache, so the .so travels with gpurun).

    python -m paper_1806_06467_b200.build [--force]

One object per grid size N (pass_inst.cu compiled with -DFR_N=N) plus the API object; compiled in
parallel, linked into paper_1806_06467_b200/libfresnel.so.
"""
from __future__ import annotations

import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build", os.environ.get("FRESNEL_LIB_NAME", "libfresnel.so").replace(".so", ""))
# FRESNEL_LIB_NAME / FRESNEL_DEFINES: tuning builds only (e.g. FRESNEL_DEFINES="-DFR_COLW_F64=4")
LIB = os.path.join(HERE, os.environ.get("FRESNEL_LIB_NAME", "libfresnel.so"))
EXTRA_DEFINES = os.environ.get("FRESNEL_DEFINES", "").split()
SIZES = (64, 128, 256, 512, 1024, 2048, 4096, 8192)
# grid sizes of the register-resident mixed-radix pass (mr_kernel.cuh; keep in step with FR_MR_SIZES of csrc/dispatch.h)
MR_SIZES = (700, 1000, 1200, 1400, 1500, 2000, 2400, 2800, 3000, 3600, 4000, 5000, 5600, 6000)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _sources_digest() -> str:
    h = hashlib.sha256()
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for name in sorted(os.listdir(root)):
            if name.endswith((".cu", ".cuh", ".h")):
                with open(os.path.join(root, name), "rb") as fh:
                    h.update(name.encode())
                    h.update(fh.read())
    h.update(" ".join(NVCC_FLAGS + EXTRA_DEFINES).encode())
    return h.hexdigest()


def _compile(args):
    src, obj, extra = args
    cmd = [_nvcc(), *NVCC_FLAGS, *EXTRA_DEFINES, *extra, "-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed: {' '.join(cmd)}\n{r.stdout}\n{r.stderr}")
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "digest.txt")
    digest = _sources_digest()
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == digest:
        return LIB
    jobs = [(os.path.join(CSRC, "fresnel_api.cu"), os.path.join(OBJ, "fresnel_api.o"), [])]
    # the longest compilations first (the shared-memory pass: ~75 k instructions per instantiation)
    for f64 in (1, 0):
        for nt in (256, 512):
            jobs.append((os.path.join(CSRC, "gen_inst.cu"), os.path.join(OBJ, f"gen_{'f64' if f64 else 'f32'}_{nt}.o"),
                         [f"-DFR_GEN_F64={f64}", f"-DFR_GEN_NT={nt}"]))
    jobs.append((os.path.join(CSRC, "gen_inst.cu"), os.path.join(OBJ, "gen_inst.o"), []))
    jobs.append((os.path.join(CSRC, "mr_inst.cu"), os.path.join(OBJ, "mr_inst.o"), []))
    for n in MR_SIZES:
        jobs.append((os.path.join(CSRC, "mr_inst.cu"), os.path.join(OBJ, f"mr_{n}.o"), [f"-DFR_MR_N={n}"]))
    for n in SIZES:
        jobs.append((os.path.join(CSRC, "pass_inst.cu"), os.path.join(OBJ, f"pass_{n}.o"), [f"-DFR_N={n}"]))
    with cf.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(_compile, jobs))
    cmd = [_nvcc(), "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed: {' '.join(cmd)}\n{r.stdout}\n{r.stderr}")
    with open(stamp, "w") as fh:
        fh.write(digest)
    if verbose:
        print("built", LIB)
    return LIB


def build_microbench() -> str:
    """The stand-alone roof measurements of csrc/microbench.cu (HBM copy, DFMA/FFMA rates, in-SM rates of the
    transform code): the numbers bench.py's `roofline.alu` and DESIGN.md quote (profiles/r01_microbench.txt)."""
    out = os.path.join(HERE, "microbench")
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "--expt-relaxed-constexpr",
           "-o", out, os.path.join(CSRC, "microbench.cu")]
    subprocess.run(cmd, check=True)
    return out


if __name__ == "__main__":
    if "--microbench" in sys.argv:
        print("built", build_microbench())
    else:
        build(force="--force" in sys.argv, verbose=True)
