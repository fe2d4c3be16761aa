"""Builds libetp.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libetp.so")
SOURCES = ["etp_plan.cpp", "etp_eplb.cpp", "etp_lower.cpp", "etp_validate.cpp", "etp_lower_dev.cu", "etp_copy.cu", "etp_copy_static.cu", "etp_exec.cu", "etp_linear.cu", "etp_linear_group.cu", "etp_moe.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC,-Wall",
         "-I", os.path.join(ROOT, "include"), "-I", CSRC]


# debug build: ETP_BOUNDED_WAITS=1 in the environment also bounds the mbarrier waits of the tcgen05 kernels (csrc/etp_wait.cuh; kernel (a)'s are always bounded)
if os.environ.get("ETP_BOUNDED_WAITS"):
    FLAGS = FLAGS + ["-DETP_BOUNDED_WAITS=" + os.environ["ETP_BOUNDED_WAITS"]]


def _stale() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "etp.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return SO
    objs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    procs = []
    for src in SOURCES:
        obj = os.path.join(HERE, "build", src.rsplit(".", 1)[0] + ".o")
        cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-x", "cu", "-dc" if False else "-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{out}")
        if verbose and out:
            print(out)
    cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", SO] + objs
    subprocess.check_call(cmd)
    return SO


def kernel_sass_sha(pattern: str = "etp_interval_copy_kernel", so: str = SO) -> str:
    """sha256 (first 16 hex digits) of the SASS instruction text of every function of the built library whose mangled name
    contains ``pattern`` (cuobjdump -sass; addresses and encodings stripped).  It stamps an ncu capture with the exact
    kernel it profiled: bench.py reports it beside ``roofline.traffic`` and a CPU test fails when the built kernel no longer
    matches the capture under profiles/."""
    import hashlib
    import re
    cuobjdump = os.path.join(os.path.dirname(NVCC), "cuobjdump")
    out = subprocess.run([cuobjdump, "-sass", so], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, check=True).stdout
    h = hashlib.sha256()
    take, n = False, 0
    ins = re.compile(r"^\s*/\*[0-9a-f]{4,}\*/\s+(.*?;)")
    for line in out.splitlines():
        if "Function :" in line:
            take = pattern in line
            continue
        if take:
            m = ins.match(line)
            if m:
                h.update(" ".join(m.group(1).split()).encode() + b"\n")
                n += 1
    if n == 0:
        raise RuntimeError(f"no SASS found for a function matching {pattern!r} in {so}")
    return h.hexdigest()[:16]


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
