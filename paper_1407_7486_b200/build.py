"""Builds csrc/*.cu into paper_1407_7486_b200/libwl.so with nvcc for sm_100a (in-tree).

    python -m paper_1407_7486_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  cudart is linked statically so the library has no
run-time dependency on a particular libcudart.so (it shares the primary context, and so
device pointers and streams, with PyTorch in the same process).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
LIB = os.path.join(HERE, "libwl.so")
SOURCES = ("wl_api.cu", "wl_host.cu", "wl_eval_kernels.cu", "wl_wilson_sech2_f32.cu", "wl_wilson_sech2_f64.cu", "wl_wilson_fluxtube_f32.cu", "wl_generate_finalize.cu", "wl_action.cu", "wl_eval_static.cu", "wl_pipe_probe.cu")
HEADERS = ("wl_internal.cuh", "wl_field_device.cuh", "wl_dloop_device.cuh", "wl_wilson_body.cuh", "wl_terms_generic.cuh",
           "wl_terms_packed_f32.cuh", "wl_terms_sech2_f64.cuh", "wl_block_bounds.cuh")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-cudart", "static",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(INCLUDE, "wl.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = _nvcc()
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src[:-3] + ".o")
        cmd = [nvcc] + NVCC_FLAGS + os.environ.get("WL_EXTRA_NVCC_FLAGS", "").split() + [
            "-I", INCLUDE, "-I", CSRC, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode != 0:
            sys.stderr.write(out)
        if p.returncode != 0:
            raise RuntimeError("nvcc failed on %s" % src)
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a",
           "-Xcompiler", "-fPIC", "-o", tmp] + objs
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
