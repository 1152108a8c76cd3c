"""Build csrc/*.cu into libgridff.so for sm_100a with nvcc (cross-compiles without a GPU).

    python -m paper_2508_15522_b200.csrc.build [--force] [--stress]

--stress also builds libgridff_stress.so: the same sources with -DGRIDFF_STRESS (pseudo-random per-lane delays around every synchronisation
point, gridff_internal.cuh); tests/test_gpu_stress.py compares it with the product library bit for bit.  The product never loads it.
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libgridff.so")
LIB_STRESS = os.path.join(HERE, "libgridff_stress.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--threads", "4"]


def sources():
    return sorted(glob.glob(os.path.join(HERE, "*.cu")))


def stale(lib=LIB):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = sources() + glob.glob(os.path.join(HERE, "*.cuh")) + [os.path.join(HERE, "..", "..", "include", "gridff.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build_stress(force=False):
    return build(force=force, stress=True)


def build(force=False, verbose=False, stress=False):
    lib = LIB_STRESS if stress else LIB
    if not force and not stale(lib):
        return lib
    objs = []
    procs = []
    for src in sources():
        obj = src[:-3] + (".stress.o" if stress else ".o")
        objs.append(obj)
        procs.append((src, subprocess.Popen([NVCC] + FLAGS + (["-DGRIDFF_STRESS"] if stress else []) + ["-c", src, "-o", obj],
                                            stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    log = []
    for src, p in procs:
        out, _ = p.communicate()
        log.append(out)
        if p.returncode != 0:
            sys.stderr.write(out)
            raise RuntimeError("nvcc failed on %s" % src)
    subprocess.check_call([NVCC, "-shared", "-o", lib] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
    with open(os.path.join(HERE, "build_stress.log" if stress else "build.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--stress" in sys.argv:
        print(build(force="--force" in sys.argv, stress=True))
