"""Compile libltvscan.so (sm_100a only) in-tree with nvcc.  `python -m paper_2606_14188_b200.build`."""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libltvscan.so")
SOURCES = ["api.cu", "rollout.cu", "adjoint.cu", "phi.cu", "phi_simt.cu", "phi_tc.cu", "kalman.cu", "constraints.cu", "riccati_scan.cu", "output_feedback.cu", "fused_small.cu", "kalman_small.cu", "no_alloc.cu", "assemble.cu", "margins.cu", "phi_rows.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
    "--expt-relaxed-constexpr",
    "-cudart", "static",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libltvscan.so cannot be built (there is no CPU fallback)")


STAMP = LIB + ".srchash"


def source_hash() -> str:
    """sha256 over the content of every file the library is built from (csrc/*, include/ltv_scan.h), this script, the nvcc
    flags and the nvcc version.  Stored beside the .so at build time: a pushed binary whose sources have since changed is
    rebuilt whatever the file times say."""
    import hashlib

    h = hashlib.sha256()
    deps = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC))
    deps += [os.path.normpath(os.path.join(HERE, "..", "include", "ltv_scan.h")), os.path.abspath(__file__)]
    for d in deps:
        h.update(os.path.basename(d).encode() + b"\0")
        with open(d, "rb") as f:
            h.update(f.read())
    h.update(" ".join(NVCC_FLAGS + SOURCES).encode())
    h.update(os.environ.get("LTV_SCAN_NVCC_EXTRA", "").encode())
    try:
        h.update(subprocess.run([_nvcc(), "--version"], capture_output=True, text=True).stdout.encode())
    except Exception:
        pass
    return h.hexdigest()


def _stale() -> bool:
    if not (os.path.exists(LIB) and os.path.exists(STAMP)):
        return True
    with open(STAMP) as f:
        return f.read().strip() != source_hash()


def build(force: bool = False, verbose: bool = False) -> str:
    """Build the shared library unless the one in place was built from exactly these sources and flags (content hash,
    not file times); returns its path."""
    if not force and not _stale():
        return LIB
    want = source_hash()
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    nvcc = _nvcc()
    objs, procs = [], []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, *os.environ.get("LTV_SCAN_NVCC_EXTRA", "").split(), "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    failed = False
    for src, pr in procs:
        out, _ = pr.communicate()
        if pr.returncode != 0 or verbose:
            sys.stderr.write(f"--- nvcc {src}\n{out}\n")
        failed |= pr.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    cmd = [nvcc, "-shared", "-cudart", "static", "-o", LIB + ".tmp", *objs, "-Xlinker", "--exclude-libs,ALL"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    with open(STAMP, "w") as f:
        f.write(want + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
