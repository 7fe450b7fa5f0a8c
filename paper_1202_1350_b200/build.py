"""Build step: nvcc -> paper_1202_1350_b200/libvc.so (sm_100a only, in-tree so it travels with gpurun)."""
from __future__ import annotations

import os
import subprocess
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
SO = HERE / "libvc.so"
SOURCES = ["vc_api.cu", "vc_fused.cu", "vc_hosted.cu", "vc_verify.cu", "vc_verify_gpu.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def nvcc() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    raise RuntimeError("nvcc not found")


def newest_source_mtime() -> float:
    files = list(CSRC.glob("*")) + [HERE.parent / "include" / "vc.h"]
    return max(f.stat().st_mtime for f in files)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and SO.exists() and SO.stat().st_mtime >= newest_source_mtime():
        return SO
    tmp = SO.with_suffix(f".tmp{os.getpid()}.so")
    extra = os.environ.get("VC_NVCC_EXTRA", "").split()      # e.g. -DVC_TRACE / -DVC_POISON debug builds
    cmd = [nvcc()] + NVCC_FLAGS + extra + ["-o", str(tmp)] + [str(CSRC / s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(" ".join(cmd))
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed")
    (HERE / "ptxas.log").write_text(res.stderr)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
