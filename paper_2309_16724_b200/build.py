"""Build step: compiles the CUDA kernels + C-ABI into paper_2309_16724_b200/libsu2heff.so
(in-tree, sm_100a) with nvcc.  Used by __graft_entry__.build() and by `python -m
paper_2309_16724_b200.build`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SOURCES = ["plan.cpp", "tensor_maps.cpp", "kernels.cu", "heff_tma.cu", "heff_small.cu", "davidson.cu", "gemm_pair.cu", "gemm_pair_small.cu", "precontract.cu", "renorm.cu", "apply_noalloc.cu"]
LIB = os.path.join(HERE, "libsu2heff.so")
PROBE_LIB = os.path.join(HERE, "libsu2probe.so")      # measurement aid of bench.py (include/su2_probe.h), not the product


def _stale():
    if not os.path.exists(LIB) or not os.path.exists(PROBE_LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(HERE, "csrc", f) for f in os.listdir(os.path.join(HERE, "csrc"))]
    deps.append(os.path.join(ROOT, "include", "su2_heff.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC", "-shared", "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(HERE, "csrc")]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(HERE, "csrc", s) for s in SOURCES] + ["-o", LIB]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libsu2heff.so")
    if verbose:
        sys.stderr.write(res.stderr)
    res = subprocess.run(cmd[:cmd.index("-shared") + 1] + ["-I" + os.path.join(ROOT, "include"),
                          os.path.join(HERE, "csrc", "peak_probe.cu"), "-o", PROBE_LIB], capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libsu2probe.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
