"""Build the CPU oracle (test infrastructure) beside its source: oracle/libvroracle.so."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(HERE, "libvroracle.so")
SRC = os.path.join(HERE, "vr_oracle.c")


def build(force=False):
    if force or not os.path.exists(SO) or os.path.getmtime(SRC) > os.path.getmtime(SO):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", SO, SRC, "-lm"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("oracle build failed: %s\n%s" % (" ".join(cmd), r.stderr))
    return SO


if __name__ == "__main__":
    print(build(force=True))
