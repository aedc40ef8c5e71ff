"""Build libfh_b200.so (the C-ABI library) in-tree with nvcc for sm_100a."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfh_b200.so")
SOURCES = ["zgemm.cu", "zgemm_ws.cu", "zgemm_tc.cu", "kernels.cu", "api.cu", "tdvp.cu", "noalloc.cu", "symmetry.cpp", "su2.cpp"]
HEADERS = ["fh_internal.hpp", "symmetry.hpp", "context.hpp"]


def source_digest():
    """Hash of every source, header and compile flag that goes into the library."""
    import hashlib
    h = hashlib.sha256()
    for f in SOURCES + HEADERS:
        h.update(open(os.path.join(CSRC, f), "rb").read())
    h.update(open(os.path.join(ROOT, "include", "fh_b200.h"), "rb").read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]
STAMP = os.path.join(HERE, "build", "libfh_b200.sha256")


def build(force=False, verbose=False):
    """Compile every CUDA / C++ source for sm_100a and link libfh_b200.so in-tree.  The library is rebuilt unless
    a stamp written by THIS build procedure says that the .so on disk was made from exactly the present sources
    and flags (a .so that merely looks newer than the sources, e.g. one shipped from another machine, is not
    trusted)."""
    digest = source_digest()
    if not force and os.path.exists(LIB) and os.path.exists(STAMP) and open(STAMP).read().strip() == digest:
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    procs = []
    for src in SOURCES:
        obj = os.path.join(HERE, "build", src + ".o")
        cmd = [nvcc] + NVCC_FLAGS + ["-x", "cu", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
                                     "-c", os.path.join(CSRC, src), "-o", obj]
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
    cmd = [nvcc, "-shared", "-o", LIB] + objs + ["-L/usr/local/cuda/lib64", "-lcusolver", "-lcublas",
                                                  "-Xlinker", "-rpath=/usr/local/cuda/lib64"]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stdout)
    with open(STAMP, "w") as f:
        f.write(digest + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
