"""Build libesc.so (the C-ABI library of include/esc.h) in-tree with nvcc for sm_100a.

Run: python -m paper_2606_20537_b200.build [--force] [--verbose]
The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
SOURCES = ["esc_host.cu", "copy_kernel.cu", "stage.cu", "scan_api.cu", "scan_kernel.cu", "gdn_kernel.cu", "gdn_scan_kernel.cu", "graph.cu", "noalloc.cu"]
HEADERS = [os.path.join(ROOT, "include", "esc.h"), os.path.join(CSRC, "esc_internal.h"), os.path.join(CSRC, "sm100_ptx.cuh")]
TARGET = os.path.join(PKG, "libesc.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-DESC_BUILD",] + (["-DESC_TC_TRACE"] if os.environ.get("ESC_TC_TRACE") else []) + (["-DESC_SCAN_PROF"] if os.environ.get("ESC_SCAN_PROF") else []) + (["-DESC_GDN_PROF"] if os.environ.get("ESC_GDN_PROF") else []) + (["-D" + x for x in os.environ.get("ESC_DEFS", "").split()]) + (["-DESC_MBAR_BACKOFF=" + os.environ["ESC_MBAR_BACKOFF"]] if os.environ.get("ESC_MBAR_BACKOFF") else []) + [
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]


def _nvcc():
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(TARGET):
        return True
    t = os.path.getmtime(TARGET)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return TARGET
    objs = []
    bdir = os.path.join(PKG, "build")
    os.makedirs(bdir, exist_ok=True)
    procs = []
    for s in SOURCES:
        obj = os.path.join(bdir, s.replace(".cu", ".o"))
        objs.append(obj)
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, s), "-o", obj]
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for s, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write("== %s ==\n%s\n" % (s, out))
        failed = failed or p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    tmp = TARGET + ".tmp.%d" % os.getpid()
    subprocess.run([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp] + objs, check=True)
    os.replace(tmp, TARGET)
    return TARGET


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
