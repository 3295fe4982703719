"""Build libvog.so (sm_100a) in-tree with nvcc: one object per line length, compiled in parallel.

    python -m paper_1301_5892_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so lands next to this file so it travels with the
repository snapshot to the GPU box; objects go to build/ (git-ignored).
"""
import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libvog.so")
SIZES = (64, 128, 256, 512)   # whole-line kernels; longer lines use the overlap-save kernels (vog_os.cu)
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "--use_fast_math=false"]
FLAGS = [f for f in FLAGS if f != "--use_fast_math=false"]


def _sources():
    out = []
    for root, _d, files in os.walk(CSRC):
        out += [os.path.join(root, f) for f in files]
    out.append(os.path.join(os.path.dirname(HERE), "include", "vog.h"))
    return out


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(job):
    src, obj, extra = job
    cmd = [NVCC] + FLAGS + extra + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return obj


def build(force=False, verbose=False):
    deps = _sources()
    if not force and not _stale(LIB, deps):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    jobs = [(os.path.join(CSRC, "vog_lib.cu"), os.path.join(OBJ, "vog_lib.o"), []),
            (os.path.join(CSRC, "vog_os.cu"), os.path.join(OBJ, "vog_os.o"), []),
            (os.path.join(CSRC, "vog_stencil.cu"), os.path.join(OBJ, "vog_stencil.o"), []),
            (os.path.join(CSRC, "vog_f64.cu"), os.path.join(OBJ, "vog_f64.o"), []),
            (os.path.join(CSRC, "vog_noalloc.cu"), os.path.join(OBJ, "vog_noalloc.o"), []),
            (os.path.join(CSRC, "vog_small.cu"), os.path.join(OBJ, "vog_small.o"), [])]
    for n in SIZES:
        jobs.append((os.path.join(CSRC, "vog_advect_inst.cu"), os.path.join(OBJ, "vog_advect_%d.o" % n),
                     ["-DVOG_N=%d" % n]))
    todo = [j for j in jobs if force or _stale(j[1], deps)]
    with cf.ThreadPoolExecutor(max_workers=min(len(todo) or 1, os.cpu_count() or 4)) as ex:
        for obj in ex.map(_compile, todo):
            if verbose:
                print("built", obj)
    cmd = [NVCC, "-shared", "-o", LIB] + [j[1] for j in jobs] + ["-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
