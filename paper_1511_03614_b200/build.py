"""Build libfiesta_b200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo).

    python -m paper_1511_03614_b200.build [--force]

Objects are rebuilt only when a source or header under csrc/ or include/ is newer.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libfiesta_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVFLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + ARCH
CPLX_DIMS = range(1, 9)


def _deps():
    out = []
    for d in (CSRC, os.path.join(ROOT, "include")):
        for f in os.listdir(d):
            if f.endswith((".h", ".hpp", ".cuh", ".inc")):
                out.append(os.path.join(d, f))
    return out


def _stale(target, srcs):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in srcs)


def _run(cmd, log):
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout)
    if r.returncode != 0:
        raise RuntimeError("build step failed: %s\n%s" % (" ".join(cmd), r.stdout[-4000:]))


def build(force=False, verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    gen_src = os.path.join(CSRC, "gen_interp_ptx.py")
    gen_out = os.path.join(CSRC, "fx_interp_gen.inc")
    if force or _stale(gen_out, [gen_src, os.path.join(CSRC, "fx_isa.h")]):
        text = subprocess.run([sys.executable, gen_src], stdout=subprocess.PIPE, check=True, text=True).stdout
        with open(gen_out, "w") as f:
            f.write(text)
    hdrs = _deps()
    jobs = []  # (object, cmd, sources)

    def cu(name, src, extra=()):
        o = os.path.join(OBJ, name + ".o")
        s = os.path.join(CSRC, src)
        jobs.append((o, [NVCC] + NVFLAGS + list(extra) + ["-c", s, "-o", o], [s] + hdrs))

    cu("fx_kernels_real", "fx_kernels_real.cu")
    cu("fx_kernels_small", "fx_kernels_small.cu")
    for n in CPLX_DIMS:
        cu("fx_kernels_cplx_n%d" % n, "fx_kernels_cplx.cu", ["-DFX_N=%d" % n])
    for name in ("fiesta_abi", "fx_compiler"):
        o = os.path.join(OBJ, name + ".o")
        s = os.path.join(CSRC, name + ".cpp")
        jobs.append((o, ["g++", "-O2", "-std=c++17", "-fPIC", "-pthread", "-I/usr/local/cuda/include", "-c", s, "-o", o],
                     [s] + hdrs))
    todo = [(o, c) for (o, c, srcs) in jobs if force or _stale(o, srcs)]
    if verbose and todo:
        print("building %d objects" % len(todo), file=sys.stderr)
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
        list(ex.map(lambda oc: _run(oc[1], oc[0] + ".log"), todo))
    objs = [o for (o, _, _) in jobs]
    if force or todo or _stale(LIB, objs):
        _run([NVCC, "-shared", "-o", LIB] + ARCH + objs + ["-lcudart", "-lpthread"], os.path.join(OBJ, "link.log"))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
