"""Build paper_1807_01971_b200/libfx.so in-tree: nvcc for sm_100a (+ g++/libquadmath for the host tables).

No torch extension machinery: the library is a plain C-ABI shared object (include/fx.h) loaded with ctypes.
-fmad=false: contraction is forbidden, every FMA in the sources is explicit (footnote P:206).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libfx.so")
BUILD = os.path.join(HERE, "build")

NVCC_FLAGS = [("-D%s=%s" % (k, os.environ[k])) for k in ("FX_PFD", "FX_K1_R", "FX_K1_W", "FX_AP_R", "FX_AP_W", "FX_NBX3", "FX_MINB3", "FX_DGT_DEBUG", "FX_K1T_NS", "FX_K1T_R", "FX_K1T_NBX", "FX_K1T_ND", "EX_KL", "FX_K1_K", "FX_K1_WB", "FX_K1_KL", "FX_PERSIST_PROF", "FX_NBX1", "FX_NBX4", "FX_NBX5", "FX_MINB4", "FX_MINB5", "FX_NS5", "FX_KEEPP", "FX_K2_NODOT", "FX_CHECKED", "FX_HPAD", "FX_XVEC", "FX_EX_SKIP") if os.environ.get(k)] + ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math", "-Xptxas", "-v"]


def _sources():
    cu = sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))
    cpp = sorted(f for f in os.listdir(CSRC) if f.endswith(".cpp"))
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "fx.h"), __file__]
    return cu, cpp, deps


def build(force=False, verbose=False):
    cu, cpp, deps = _sources()
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(d) for d in deps):
        return SO
    os.makedirs(BUILD, exist_ok=True)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    log = []

    def _nvcc(f):
        o = os.path.join(BUILD, f + ".o")
        r = subprocess.run([nvcc] + NVCC_FLAGS + ["-c", os.path.join(CSRC, f), "-o", o], capture_output=True, text=True)
        return f, o, r

    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=min(len(cu), os.cpu_count() or 1)) as ex:      # one nvcc per translation unit, side by side
        for f, o, r in ex.map(_nvcc, cu):
            log.append(r.stderr)
            if r.returncode != 0:
                raise RuntimeError("nvcc failed on %s:\n%s" % (f, r.stderr))
            objs.append(o)
    for f in cpp:
        o = os.path.join(BUILD, f + ".o")
        r = subprocess.run(["g++", "-O2", "-std=gnu++17", "-fPIC", "-ffp-contract=off", "-fno-fast-math", "-c",
                            os.path.join(CSRC, f), "-o", o], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("g++ failed on %s:\n%s" % (f, r.stderr))
        objs.append(o)
    r = subprocess.run([nvcc, "-shared", "-o", SO + ".tmp"] + objs + ["-lquadmath", "-cudart", "static"],
                       capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n%s" % r.stderr)
    os.replace(SO + ".tmp", SO)
    with open(os.path.join(BUILD, "ptxas.log"), "w") as fh:
        fh.write("\n".join(log))
    if verbose:
        sys.stderr.write("\n".join(log))
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
