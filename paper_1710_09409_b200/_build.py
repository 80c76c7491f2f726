"""Compile csrc/*.cu into the in-tree libsu3stream.so for sm_100a (nvcc cross-compiles without a GPU).  The
template instantiations are spread over several translation units, compiled in parallel and linked into one
shared library.  The .so is git-ignored but travels to the GPU box with the snapshot."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
UNITS = ["su3_api", "su3_k_stream_f64", "su3_k_stream_f32", "su3_k_menu_f64", "su3_k_menu_f32", "su3_k_shiftpipe",
         "su3_k_shift", "su3_k_misc"]
SOURCES = [os.path.join(CSRC, u + ".cu") for u in UNITS]
DEPS = SOURCES + [os.path.join(CSRC, "su3_kernels.cuh"), os.path.join(CSRC, "su3_tables.h"),
                  os.path.join(os.path.dirname(HERE), "include", "su3stream.h")]
LIB = os.path.join(HERE, "libsu3stream.so")
OBJDIR = os.path.join(HERE, "build")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]


def stale() -> bool:
    return not os.path.exists(LIB) or any(os.path.getmtime(LIB) < os.path.getmtime(d) for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        os.makedirs(OBJDIR, exist_ok=True)
        pid = os.getpid()
        objs = [os.path.join(OBJDIR, "%s.%d.o" % (u, pid)) for u in UNITS]
        procs = [subprocess.Popen([NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", o, src])
                 for o, src in zip(objs, SOURCES)]
        rcs = [pr.wait() for pr in procs]
        if any(rcs):
            raise subprocess.CalledProcessError(max(rcs), NVCC)
        tmp = LIB + ".%d.tmp" % pid
        subprocess.check_call([NVCC] + FLAGS[:2] + ["-shared", "-cudart", "static", "-o", tmp] + objs)
        os.replace(tmp, LIB)
        for o in objs:
            os.remove(o)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
