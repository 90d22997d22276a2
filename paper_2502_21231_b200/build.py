"""Build csrc/libbytescale_attn.so (nvcc, sm_100a only) and the host-only synth generator.

    python -m paper_2502_21231_b200.build [--force]

The library links the CUDA runtime statically and nothing else (the driver entry point for TMA
tensor maps is resolved at run time), so it loads on a machine without a GPU; only calls that
launch kernels need one.  Built in-tree so that the .so travels with the repository snapshot.
"""
import concurrent.futures
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
SO = os.path.join(CSRC, "libbytescale_attn.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-I", CSRC] + \
    os.environ.get("BS_NVCC_EXTRA", "").split()  # e.g. -DBS_FWD_EMU=0 for kernel experiments


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cpp")))


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    srcs = sources()
    hdrs = glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(ROOT, "include", "*.h"))
    objdir = os.path.join(CSRC, "build")
    os.makedirs(objdir, exist_ok=True)
    jobs = []
    for s in srcs:
        o = os.path.join(objdir, os.path.basename(s) + ".o")
        if force or _stale(o, [s] + hdrs):
            extra = ["-Xptxas", "-v"] if verbose else []
            jobs.append((s, o, [NVCC] + FLAGS + extra + ["-x", "cu", "-c", s, "-o", o]))
    with concurrent.futures.ThreadPoolExecutor(max_workers=8) as ex:
        futs = {ex.submit(subprocess.run, cmd, capture_output=True, text=True): (s, cmd)
                for s, o, cmd in jobs}
        for f in concurrent.futures.as_completed(futs):
            r = f.result()
            if verbose or r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode != 0:
                raise RuntimeError("nvcc failed on " + futs[f][0])
    objs = [os.path.join(objdir, os.path.basename(s) + ".o") for s in srcs]
    if force or jobs or _stale(SO, objs):
        subprocess.check_call([NVCC, "-shared", "-cudart", "static", "-o", SO] + objs)
    from .synth import rng
    rng.build(force)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
