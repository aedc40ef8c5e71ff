"""Build libfh_b200.so (the C-ABI library) in-tree with nvcc for sm_100a."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfh_b200.so")
SOURCES = ["zgemm.cu", "zgemm_ws.cu", "kernels.cu", "api.cu", "tdvp.cu", "symmetry.cpp", "su2.cpp"]
HEADERS = ["fh_internal.hpp", "symmetry.hpp", "context.hpp"]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(ROOT, "include", "fh_b200.h")]
    return any(os.path.getmtime(d) > t for d in deps)


TRACE_LIB = os.path.join(HERE, "libfh_b200_trace.so")


def build(force=False, verbose=False, trace=False):
    """trace=True builds libfh_b200_trace.so instead: the same library with -DFH_UNIT_TRACE (every GEMM unit
    stamps its begin/end time, SM and warp slot; used by unit_timeline.py, never by tests or bench)."""
    lib = TRACE_LIB if trace else LIB
    if not trace and not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    procs = []
    for src in SOURCES:
        obj = os.path.join(HERE, "build", src + (".trace.o" if trace else ".o"))
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
               "-Xcompiler", "-fPIC", "-x", "cu", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
               "-c", os.path.join(CSRC, src), "-o", obj]
        if trace:
            cmd.insert(1, "-DFH_UNIT_TRACE")
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s" % (src, out))
        if verbose and out:
            print(out)
    cmd = [nvcc, "-shared", "-o", lib] + objs + ["-L/usr/local/cuda/lib64", "-lcusolver", "-lcublas",
                                                  "-Xlinker", "-rpath=/usr/local/cuda/lib64"]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stdout)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv))
