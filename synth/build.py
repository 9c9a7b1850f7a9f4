"""Build the input-generator libraries beside their sources.

  libvrsynth_cpu.so   gcc   vr_synth_cpu.c   (host evaluator, table builder)
  libvrsynth_cuda.so  nvcc  vr_synth_cuda.cu (device twin, sm_100a)

Both are rebuilt only when older than their sources. nvcc cross-compiles without a GPU.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CPU_SO = os.path.join(HERE, "libvrsynth_cpu.so")
CUDA_SO = os.path.join(HERE, "libvrsynth_cuda.so")


def _stale(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("build failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))


def build_cpu(force=False):
    src = [os.path.join(HERE, "vr_synth_cpu.c"), os.path.join(HERE, "vr_synth.h")]
    if force or _stale(CPU_SO, src):
        _run(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-mfma", "-fopenmp", "-shared", "-fPIC",
              "-o", CPU_SO, src[0], "-lm"])
    return CPU_SO


def build_cuda(force=False):
    src = [os.path.join(HERE, "vr_synth_cuda.cu"), os.path.join(HERE, "vr_synth.h")]
    if force or _stale(CUDA_SO, src):
        _run(["nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-fmad=false", "-shared", "-Xcompiler", "-fPIC", "-o", CUDA_SO, src[0]])
    return CUDA_SO


def build(force=False):
    build_cpu(force)
    build_cuda(force)


if __name__ == "__main__":
    build(force=True)
    print(CPU_SO)
    print(CUDA_SO)
