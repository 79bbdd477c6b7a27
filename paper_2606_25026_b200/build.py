"""Build libwdm.so (sm_100a) in-tree with nvcc: wdm.cu + wdm_particles.cu + one object of wdm_sweeps.cu
per supported (dtype, N).  `python -m paper_2606_25026_b200.build [--force]`."""
from __future__ import annotations

import os
import re
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
# WDM_BUILD_DIR / WDM_LIB_OUT / WDM_NVCC_FLAGS: a second build beside the product's (developer A/B runs of a compile-time switch)
OBJ = os.environ.get("WDM_BUILD_DIR", os.path.join(HERE, "build"))
LIB = os.environ.get("WDM_LIB_OUT", os.path.join(HERE, "libwdm.so"))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
         "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC"]


def _sizes():
    """(dtype, N) pairs listed in wdm_plan.hpp's factorisation tables."""
    text = open(os.path.join(CSRC, "wdm_plan.hpp")).read()
    out = []
    for dtype, name in ((0, "WDM_FACT_C64"), (1, "WDM_FACT_C128")):
        body = text.split(f"#define {name}(X)")[1].split("#define")[0].split("inline")[0]
        out += [(dtype, int(n)) for n in re.findall(r"X\((\d+),", body)]
    return out


def _newest_source() -> float:
    inc = os.path.join(HERE, "..", "include")
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(inc, f) for f in os.listdir(inc)]
    return max(os.path.getmtime(f) for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    newest = _newest_source()
    jobs = [("wdm.o", ["-c", os.path.join(CSRC, "wdm.cu")]),
            ("wdm_particles.o", ["-c", os.path.join(CSRC, "wdm_particles.cu")]),
            ("wdm_dist.o", ["-c", os.path.join(CSRC, "wdm_dist.cu")])]
    for dtype, n in _sizes():
        jobs.append((f"sweeps_{dtype}_{n}.o", [f"-DWDM_DTYPE={dtype}", f"-DWDM_N={n}", "-c", os.path.join(CSRC, "wdm_sweeps.cu")]))

    def run(job):
        name, args = job
        out = os.path.join(OBJ, name)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= newest:
            return out
        cmd = [NVCC, *FLAGS, *os.environ.get("WDM_NVCC_FLAGS", "").split(), *(["-Xptxas", "-v"] if verbose else []), *args, "-o", out]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {name}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
        return out

    with ThreadPoolExecutor(max_workers=max(1, (os.cpu_count() or 2))) as ex:
        objs = list(ex.map(run, jobs))
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        r = subprocess.run([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs],
                           capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
