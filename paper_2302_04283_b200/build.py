"""Build librad.so (hand-written CUDA for sm_100a + host C++) in-tree with nvcc.

    python -m paper_2302_04283_b200.build [--force]

nvcc cross-compiles without a GPU.  The library is written next to this file so that it
travels with the source tree to the GPU box.
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "librad.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC,-ffp-contract=off",
         "-I", os.path.join(ROOT, "include"), "-I", CSRC]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cpp")))


def _compile(args):
    src, obj, flags = args
    subprocess.check_call([NVCC] + flags + ["-c", src, "-o", obj])
    return obj


def build(force=False, verbose=False):
    """compile every source of csrc/ (in parallel, one object per file) and link librad.so next to this file"""
    deps = sources() + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(ROOT, "include", "rad.h"), os.path.abspath(__file__)]
    if not force and os.path.exists(SO) and os.path.getmtime(SO) >= max(os.path.getmtime(d) for d in deps):
        return SO
    import concurrent.futures
    import tempfile
    flags = FLAGS + (["-Xptxas", "-v"] if verbose else [])
    with tempfile.TemporaryDirectory() as tmp:
        jobs = [(s, os.path.join(tmp, os.path.basename(s) + ".o"), flags) for s in sources()]
        with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
            objs = list(ex.map(_compile, jobs))
        subprocess.check_call([NVCC] + FLAGS + ["-shared", "-o", SO] + objs)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
