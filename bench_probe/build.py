"""Build bench_probe/libsg_probe.so: the ALU-pipe (LOP3) peak micro-benchmark that bench.py runs for its roofline
denominator.  An instrument of the benchmark, not part of the product library or its ABI; built by bench.py and by
__graft_entry__.build(), never by paper_1403_4560_b200/build.py."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
PROBE_SRC = os.path.join(HERE, "alu_probe.cu")
PROBE_LIB = os.path.join(HERE, "libsg_probe.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-fmad=false",
         "-Xcompiler", "-fPIC,-O2,-Wall", "-shared"]


def build_probe(force=False):
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_LIB) < os.path.getmtime(PROBE_SRC):
        tmp = PROBE_LIB + ".tmp.%d" % os.getpid()
        subprocess.run([NVCC, *FLAGS, "-o", tmp, PROBE_SRC], check=True)
        os.replace(tmp, PROBE_LIB)
    return PROBE_LIB


if __name__ == "__main__":
    print(build_probe(force=True))
