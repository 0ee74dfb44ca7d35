"""Build libnk.so (sm_100a) in-tree with nvcc.  No torch, no JIT cache: the .so sits next to
this file so that it travels with the repository snapshot.

    python -m paper_2606_20917_b200.build [--force] [-j N]

One translation unit per (shape, P) (csrc/nk_inst.cu with -DNK_SHAPE/-DNK_P) plus the API and
the host tables; objects go to build/ and are rebuilt only when a source is newer.
"""
import argparse
import concurrent.futures as cf
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libnk.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
MAX_P = {0: 10, 1: 8, 2: 8}          # hex, tet, prism  (must match kMaxP in nk_api.cu)
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", INCLUDE]


def _nvcc():
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libnk cannot be built (there is no CPU fallback)")
    return exe


def _sources():
    return [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))] + [os.path.join(INCLUDE, "nk.h"), __file__]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return r.stdout + r.stderr


def build(force=False, jobs=None, verbose=False, extra_defs=(), lib=None, objdir=None, only=None):
    """extra_defs / lib / objdir: a tuning build (-D switches of csrc/nk_kernels.cuh) into another library file, to be
    loaded with NK_LIB=<path>; only: iterable of (shape, P) pairs to instantiate (the others keep their objects)."""
    global OBJ, LIB
    nvcc = _nvcc()
    if objdir:
        OBJ = objdir
    if lib:
        LIB = lib
    os.makedirs(OBJ, exist_ok=True)
    deps = _sources()
    jobs = jobs or max(1, (os.cpu_count() or 2))
    tasks = []
    api_o = os.path.join(OBJ, "nk_api.o")
    tasks.append((api_o, [nvcc, *COMMON, *ARCH, "-c", os.path.join(CSRC, "nk_api.cu"), "-o", api_o]))
    dense_o = os.path.join(OBJ, "nk_dense.o")
    tasks.append((dense_o, [nvcc, *COMMON, *ARCH, *(["-Xptxas", "-v"] if verbose else []), "-c",
                            os.path.join(CSRC, "nk_dense.cu"), "-o", dense_o]))
    # the text of nk_dense.cuh as a C++ raw string literal, for the NVRTC path of nk_jit.cu
    src_inc = os.path.join(OBJ, "nk_dense_src.inc")
    text = 'R"NKSRC(' + open(os.path.join(CSRC, "nk_dense.cuh")).read() + ')NKSRC"\n'
    if not os.path.exists(src_inc) or open(src_inc).read() != text:
        with open(src_inc, "w") as f:
            f.write(text)
    # the same for the sum-factorised kernel template and the stage files it includes: {name, text} pairs
    sf_inc = os.path.join(OBJ, "nk_sumfac_src.inc")
    names = ["nk_kernels.cuh", "nk_kernel_body.cuh"] + sorted(f for f in os.listdir(CSRC) if f.startswith("nk_stage_") and f.endswith(".inc"))
    text = "".join('{"%s", R"NKSRC(%s)NKSRC"},\n' % (n, open(os.path.join(CSRC, n)).read()) for n in names)
    if not os.path.exists(sf_inc) or open(sf_inc).read() != text:
        with open(sf_inc, "w") as f:
            f.write(text)
    jit_o = os.path.join(OBJ, "nk_jit.o")
    tasks.append((jit_o, [nvcc, *COMMON, *ARCH, "-I", OBJ, "-c", os.path.join(CSRC, "nk_jit.cu"), "-o", jit_o]))
    sol_o = os.path.join(OBJ, "nk_solver.o")
    tasks.append((sol_o, [nvcc, *COMMON, *ARCH, "-c", os.path.join(CSRC, "nk_solver.cu"), "-o", sol_o]))
    tab_o = os.path.join(OBJ, "nk_host_tables.o")
    tasks.append((tab_o, [nvcc, *COMMON, "-c", os.path.join(CSRC, "nk_host_tables.cpp"), "-o", tab_o]))
    for shape, pmax in MAX_P.items():
        for P in range(pmax, 0, -1):     # big orders first: they compile longest
            o = os.path.join(OBJ, "nk_inst_%d_%d.o" % (shape, P))
            cmd = [nvcc, *COMMON, *ARCH, *extra_defs, "-DNK_SHAPE=%d" % shape, "-DNK_P=%d" % P,
                   "-c", os.path.join(CSRC, "nk_inst.cu"), "-o", o]
            if verbose:
                cmd[1:1] = ["-Xptxas", "-v"]
            tasks.append((o, cmd))
    tasks.sort(key=lambda t: 0 if "inst" in t[0] else 1)
    todo = [t for t in tasks if force or _stale(t[0], deps)]
    logs = []
    if todo:
        with cf.ThreadPoolExecutor(max_workers=jobs) as ex:
            for out in ex.map(lambda t: _run(t[1]), todo):
                logs.append(out)
    objs = [t[0] for t in tasks]
    if todo or _stale(LIB, objs):
        _run([nvcc, "-shared", *ARCH, "-o", LIB, *objs, "-lcudart", "-ldl"])
    return "\n".join(logs)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("-j", type=int, default=None)
    ap.add_argument("-v", action="store_true")
    ap.add_argument("--defs", default="", help="extra -D switches, space separated (tuning builds)")
    ap.add_argument("--lib", default=None, help="output library (default: libnk.so next to this file)")
    ap.add_argument("--objdir", default=None)
    a = ap.parse_args()
    out = build(force=a.force, jobs=a.j, verbose=a.v, extra_defs=tuple(a.defs.split()), lib=a.lib, objdir=a.objdir)
    if a.v:
        sys.stdout.write(out)
    print(LIB)


if __name__ == "__main__":
    main()
