"""Build step: run the code generator, then compile every CUDA source for sm_100a into
paper_2303_18244_b200/libme_b200.so (in-tree, so it travels to the GPU box).  nvcc cross-compiles
without a GPU.  Usage: python -m paper_2303_18244_b200.build [-j N] [--force]"""
import concurrent.futures
import hashlib
import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
GEN = os.path.join(CSRC, "generated")
OBJ = os.path.join(PKG, "build")
LIB = os.path.join(PKG, "libme_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
CFLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr", "-Xptxas", "-v"]


def _digest(paths):
    h = hashlib.sha256()
    for p in sorted(paths):
        with open(p, "rb") as f:
            h.update(p.encode()); h.update(f.read())
    h.update(" ".join(CFLAGS + ARCH).encode())
    return h.hexdigest()


def _compile(src, obj, headers):
    stamp = obj + ".sha"
    dig = _digest([src] + headers)
    if os.path.exists(obj) and os.path.exists(stamp) and open(stamp).read() == dig:
        return src, "cached", ""
    cmd = [NVCC] + ARCH + CFLAGS + ["-I", CSRC, "-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, r.stdout, r.stderr))
    with open(stamp, "w") as f:
        f.write(dig)
    with open(obj + ".ptxas.txt", "w") as f:
        f.write(r.stderr)
    return src, "built", r.stderr


def build(jobs=None, force=False, verbose=False):
    from .codegen.__main__ import main as gen_main
    os.makedirs(OBJ, exist_ok=True)
    gen_main(GEN)
    srcs = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith(".cu")]
    srcs += [os.path.join(GEN, f) for f in sorted(os.listdir(GEN)) if f.endswith(".cu")]
    headers = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))]
    headers += [os.path.join(GEN, f) for f in os.listdir(GEN) if f.endswith((".h", ".cuh"))]
    headers.append(os.path.join(os.path.dirname(PKG), "include", "me.h"))
    if force:
        for f in os.listdir(OBJ):
            os.remove(os.path.join(OBJ, f))
    objs = [os.path.join(OBJ, os.path.basename(s)[:-3] + ".o") for s in srcs]
    jobs = jobs or os.cpu_count() or 4
    changed = False
    with concurrent.futures.ThreadPoolExecutor(jobs) as ex:
        for src, what, log in ex.map(lambda so: _compile(so[0], so[1], headers), zip(srcs, objs)):
            if what == "built":
                changed = True
            if verbose:
                print("[%s] %s" % (what, os.path.relpath(src, PKG)))
    if changed or not os.path.exists(LIB):
        cmd = [NVCC] + ARCH + ["-shared", "-o", LIB] + objs + ["-lcudart"]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    j = None
    if "-j" in sys.argv:
        j = int(sys.argv[sys.argv.index("-j") + 1])
    print(build(jobs=j, force="--force" in sys.argv, verbose=True))
