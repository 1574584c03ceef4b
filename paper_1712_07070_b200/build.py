"""Build libgamerhydro.so (sm_100a) in-tree with nvcc.  Usage: python -m paper_1712_07070_b200.build [--force]

One object per (scheme, recon, riemann) from csrc/inst.cu plus csrc/api.cu, compiled in parallel,
linked with the static CUDA runtime so the library loads (and exports its symbols) on a box
without a GPU.
"""
import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libgamerhydro.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "-I", CSRC]


def _sources():
    return [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh"))] + \
           [os.path.join(os.path.dirname(HERE), "include", "gamer_hydro.h")]


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return r.stdout + r.stderr


def build(force=False, verbose=False):
    newest = max(os.path.getmtime(s) for s in _sources())
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    have_ctu = os.path.exists(os.path.join(CSRC, "ctu_kernel.cuh"))
    jobs = []
    for s in (1, 2, 3):
        for r in (1, 2):
            if s == 3 and r == 2:      # VL + PPM is not built (fourth ghost zone)
                continue
            for v in (1, 2, 3, 4):
                o = os.path.join(OBJ, "inst_%d_%d_%d.o" % (s, r, v))
                cmd = [NVCC, *FLAGS, "-DG_SCHEME=%d" % s, "-DG_RECON=%d" % r, "-DG_SOLVER=%d" % v]
                if have_ctu:
                    cmd.append("-DGAMER_HAVE_CTU")
                if os.environ.get("GAMER_EXTRA_DEFS"):
                    cmd += os.environ["GAMER_EXTRA_DEFS"].split()
                if verbose:
                    cmd += ["-Xptxas", "-v"]
                jobs.append((cmd + ["-c", os.path.join(CSRC, "inst.cu"), "-o", o], o))
    for unit in ("api", "alu_peak", "noalloc"):
        o = os.path.join(OBJ, unit + ".o")
        jobs.append(([NVCC, *FLAGS, "-c", os.path.join(CSRC, unit + ".cu"), "-o", o], o))
    with concurrent.futures.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        outs = list(ex.map(lambda j: _run(j[0]), jobs))
    if verbose:
        print("\n".join(outs))
    _run([NVCC, "-shared", "-o", LIB, *[j[1] for j in jobs], "-cudart", "static"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
