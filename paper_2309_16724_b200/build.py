"""Build step: compiles the CUDA kernels + C-ABI into paper_2309_16724_b200/libsu2heff.so
(in-tree, sm_100a) with nvcc, the measurement probe into libsu2probe.so and the INT8-sliced GEMM pair
(include/su2_ozaki.h, needs the CUTLASS/CuTe header tree vendored in site-packages) into libsu2ozaki.so.
Used by __graft_entry__.build() and by `python -m paper_2309_16724_b200.build`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SOURCES = ["plan.cpp", "tensor_maps.cpp", "kernels.cu", "heff_tma.cu", "heff_two_pass.cu", "heff_small.cu", "davidson.cu", "gemm_pair.cu", "gemm_pair_small.cu", "gemm_two_pass.cu", "precontract.cu", "renorm.cu", "apply_noalloc.cu"]
LIB = os.path.join(HERE, "libsu2heff.so")
PROBE_LIB = os.path.join(HERE, "libsu2probe.so")      # measurement aid of bench.py (include/su2_probe.h), not the product
OZAKI_LIB = os.path.join(HERE, "libsu2ozaki.so")      # include/su2_ozaki.h: GEMM pair on the INT8 tensor path (row f4)
OZAKI_SOURCES = ["ozaki.cu"]


def cutlass_root():
    """The CUTLASS/CuTe header tree this image vendors (header-only; versions 4.x carry the sm_100 collective builder)."""
    env = os.environ.get("CUTLASS_ROOT")
    cands = [env] if env else []
    for sp in sys.path:
        cands += [os.path.join(sp, "flashinfer", "data", "cutlass"), os.path.join(sp, "tilelang", "3rdparty", "cutlass")]
    for c in cands:
        if c and os.path.exists(os.path.join(c, "include", "cutlass", "gemm", "collective", "collective_builder.hpp")):
            return c
    raise RuntimeError("no CUTLASS header tree found (set CUTLASS_ROOT): libsu2ozaki.so cannot be built")


def _stale():
    if not os.path.exists(LIB) or not os.path.exists(PROBE_LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(HERE, "csrc", f) for f in os.listdir(os.path.join(HERE, "csrc")) if f not in OZAKI_SOURCES]
    deps.append(os.path.join(ROOT, "include", "su2_heff.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def _ozaki_stale():
    if not os.path.exists(OZAKI_LIB):
        return True
    t = os.path.getmtime(OZAKI_LIB)
    deps = [os.path.join(HERE, "csrc", f) for f in OZAKI_SOURCES] + [os.path.join(ROOT, "include", "su2_ozaki.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build_ozaki(force=False):
    """libsu2ozaki.so: a few minutes of template instantiation, so it is rebuilt only when its own sources changed."""
    if not force and not _ozaki_stale():
        return OZAKI_LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cr = cutlass_root()
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--expt-relaxed-constexpr",
           "-Xcompiler", "-fPIC", "-shared", "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(cr, "include"),
           "-I" + os.path.join(cr, "tools", "util", "include")]
    cmd += [os.path.join(HERE, "csrc", s) for s in OZAKI_SOURCES] + ["-o", OZAKI_LIB]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libsu2ozaki.so")
    return OZAKI_LIB


def build(force=False, verbose=False):
    """All three libraries; libsu2ozaki.so (minutes of template instantiation) compiles next to the other two."""
    import concurrent.futures
    with concurrent.futures.ThreadPoolExecutor(max_workers=1) as pool:
        ozaki = pool.submit(build_ozaki, force)
        try:
            return _build_main(force, verbose)
        finally:
            ozaki.result()


def _build_main(force=False, verbose=False):
    """libsu2heff.so: every source compiled to an object file of its own, in parallel (the template-heavy kernels take up to a
    minute each), then linked; libsu2probe.so next to it."""
    if not force and not _stale():
        return LIB
    import concurrent.futures
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    flags = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
             "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(HERE, "csrc")]
    if verbose:
        flags += ["-Xptxas", "-v"]

    def compile_one(src):
        obj = os.path.join(objdir, os.path.splitext(src)[0] + ".o")
        res = subprocess.run([nvcc] + flags + ["-c", os.path.join(HERE, "csrc", src), "-o", obj], capture_output=True, text=True)
        return src, obj, res

    objs = []
    with concurrent.futures.ThreadPoolExecutor(max_workers=max(1, min(len(SOURCES), (os.cpu_count() or 2) - 1))) as pool:
        for src, obj, res in pool.map(compile_one, SOURCES):
            if res.returncode != 0:
                sys.stderr.write(res.stdout + res.stderr)
                raise RuntimeError("nvcc failed compiling %s" % src)
            if verbose:
                sys.stderr.write(res.stderr)
            objs.append(obj)
    res = subprocess.run([nvcc, "-shared", "-Xcompiler", "-fPIC"] + objs + ["-o", LIB], capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking libsu2heff.so")
    res = subprocess.run([nvcc] + flags + ["-shared", os.path.join(HERE, "csrc", "peak_probe.cu"), "-o", PROBE_LIB],
                         capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libsu2probe.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
