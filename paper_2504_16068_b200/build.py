"""In-tree build of liballegro_b200.so for sm_100a (called by __graft_entry__.build()).

Steps: (1) g++ builds the code generator csrc/gen_tp.cpp + csrc/plan.cpp and runs it, which writes
csrc/generated/tp_gen.cuh (the sparse CG table unrolled into straight-line CUDA, one set per l_max);
(2) nvcc compiles api.cu, misc.cu, model.cu, plan.cpp and inst_tp.cu / inst_env.cu once per (dtype, l_max), in
parallel; (3) nvcc links the shared library next to this file.  Nothing is cached outside the tree.

    python -m paper_2504_16068_b200.build [--force] [--jobs N]
"""
import argparse
import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
GEN = os.path.join(CSRC, "generated")
OBJ = os.path.join(HERE, "build")
INC = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "liballegro_b200.so")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
              "-I", CSRC, "-I", INC]

DTYPES = (("f32", "float"), ("f64", "double"))
LMAXS = (1, 2, 3)


def _newer(target, deps):
    if not os.path.exists(target):
        return False
    t = os.path.getmtime(target)
    return all(os.path.getmtime(d) <= t for d in deps)


def _run(cmd):
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode != 0:
        raise RuntimeError("build step failed: %s\n%s" % (" ".join(cmd), r.stdout))
    return r.stdout


def _headers():
    hs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))]
    hs.append(os.path.join(INC, "allegro_b200.h"))
    return hs


def generate(force=False):
    os.makedirs(GEN, exist_ok=True)
    os.makedirs(OBJ, exist_ok=True)
    out = os.path.join(GEN, "tp_gen.cuh")
    srcs = [os.path.join(CSRC, "gen_tp.cpp"), os.path.join(CSRC, "plan.cpp"), os.path.join(CSRC, "plan.h")]
    if not force and _newer(out, srcs):
        return out
    exe = os.path.join(OBJ, "gen_tp")
    _run(["g++", "-O2", "-std=c++17", "-o", exe, srcs[0], srcs[1]])
    _run([exe, GEN])
    return out


def _jobs():
    jobs = [("api.o", "api.cu", []), ("misc.o", "misc.cu", []), ("model.o", "model.cu", []), ("peaks.o", "peaks.cu", []), ("neighbour.o", "neighbour.cu", []), ("noalloc.o", "noalloc.cu", []), ("check.o", "check.cu", []), ("tclin.o", "tclin.cu", []), ("plan.o", "plan.cpp", [])]
    for part in (0, 1):
        jobs.insert(0, ("inst_mix3_p%d.o" % part, "inst_mix3.cu", ["-DALLEGRO_MIX3_PART=%d" % part]))
    for tag, ctype in DTYPES:
        for L in LMAXS:
            d = ["-DALLEGRO_T=%s" % ctype, "-DALLEGRO_L=%d" % L]
            jobs.append(("inst_tp_%s_l%d.o" % (tag, L), "inst_tp.cu", d))
            jobs.append(("inst_env_%s_l%d.o" % (tag, L), "inst_env.cu", d))
    # slowest files first (the pool starts jobs in list order): the l_max = 3 units, the dense l_max = 3 kernels, the tcgen05 mix
    for tag, ctype in DTYPES:
        for part in (3, 2, 1, 0):
            jobs.insert(0, ("inst_mixp_%s_p%d.o" % (tag, part), "inst_mixp.cu", ["-DALLEGRO_T=%s" % ctype, "-DALLEGRO_MIXP_PART=%d" % part]))
    slow = [j for j in jobs if j[0].startswith("inst_tp_") and j[0].endswith("_l3.o")]
    return slow + [j for j in jobs if j not in slow]


def build(force=False, jobs=None, verbose=False):
    gen = generate(force)
    deps = _headers() + [gen]
    todo, objs = [], []
    for obj, src, defs in _jobs():
        o = os.path.join(OBJ, obj)
        s = os.path.join(CSRC, src)
        objs.append(o)
        if force or not _newer(o, deps + [s]):
            todo.append(([NVCC] + NVCC_FLAGS + defs + ["-c", s, "-o", o], obj))
    if todo:
        nj = jobs or min(len(todo), os.cpu_count() or 4)
        with cf.ThreadPoolExecutor(max_workers=nj) as ex:
            futs = {ex.submit(_run, cmd): name for cmd, name in todo}
            for f in cf.as_completed(futs):
                f.result()
                if verbose:
                    print("compiled", futs[f], flush=True)
    if todo or not os.path.exists(LIB):
        tmp = LIB + ".tmp.%d" % os.getpid()
        _run([NVCC, "-shared", "-o", tmp] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--jobs", type=int, default=None)
    a = ap.parse_args()
    print(build(force=a.force, jobs=a.jobs, verbose=True))
    sys.exit(0)
