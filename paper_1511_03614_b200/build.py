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
# -fmad=false: nvcc may not contract a*b+c on its own; every FMA of the path is written as one.  The
# interpreter kernels and the native kernels (other translation units, other inlining) then do
# the same arithmetic by construction
NVFLAGS = ["-O3", "-std=c++17", "-lineinfo", "-fmad=false", "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + ARCH
CPLX_DIMS = range(1, 9)
JIT_NX = (4, 8, 12)
P_VEGAS = int(os.environ.get("FXJ_P_VEGAS", "1"))   # points per pass of the native Vegas kernels (fx_kernels.h)
# resident blocks per SM the native complex kernels are held to (register budget 65536 / (128 * blocks))
CPLX_BLOCKS = {1: 6, 2: 6, 3: 5, 4: 5, 5: 4, 6: 4, 7: 3, 8: 3}


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
    hdrs = [h for h in _deps() if not h.endswith("fx_jit_templates.inc")]
    # native tier: the evaluation kernels with the program walk left open, as PTX text per (kind,
    # dimension, mode), embedded in the library as raw strings (fx_jit.cpp splices a sector's program
    # into them)
    tpl_srcs = [os.path.join(CSRC, "fx_jit_template.cu"), os.path.join(CSRC, "fx_jit_template_cplx.cu")]
    tpl_inc = os.path.join(CSRC, "fx_jit_templates.inc")
    if force or _stale(tpl_inc, tpl_srcs + hdrs + [os.path.abspath(__file__)]):
        def fmt(n):
            return '"' + " ".join("%%%d" % i for i in range(n)) + '"'

        def ptx(job):
            cplx, n, mode = job
            out = os.path.join(OBJ, "fx_jit_template_%s%d_m%d.ptx" % ("c" if cplx else "r", n, mode))
            if cplx:
                ngh = n + n * (n + 1) // 2
                nbody = (4 if mode == 3 else (5 if mode == 2 else 4)) + 2 * n
                defs = {"FX_N": n, "FXJ_DFMT": fmt(ngh + n), "FXJ_FMT": fmt(nbody),
                        "FXJ_GH_OUTS": ", ".join('"=d"(gh[%d])' % i for i in range(ngh)),
                        "FXJ_X_INS": ", ".join('"d"(xv[%d])' % i for i in range(n)),
                        "FXJ_Z_INS": ", ".join('"d"(xv[%d]), "d"(zi[%d])' % (i, i) for i in range(n)),
                        "FXJ_CBLOCKS": CPLX_BLOCKS[n]}
                src = tpl_srcs[1]
            else:
                P = P_VEGAS if mode == 2 else 2
                nbody = (2 if mode == 3 else (2 * P + 2 if mode == 2 else P + 2)) + P * n
                defs = {"FXJ_NX": n, "FXJ_FMT": fmt(nbody), "FXJ_P_VEGAS": P_VEGAS,
                        "FXJ_XS": ", ".join('"d"(x[%d][%d])' % (k, p) for k in range(n) for p in range(P)),
                        "FXJ_WS": ", ".join('"d"(W[%d])' % p for p in range(P)),
                        "FXJ_H2S": ", ".join('"+d"(h2[%d])' % p for p in range(P))}
                src = tpl_srcs[0]
            defs["FXJ_MODE"] = mode
            hdr = out[:-4] + "_defs.h"   # operand lists contain commas: a header, not -D
            with open(hdr, "w") as f:
                f.write("".join("#define %s %s\n" % kv for kv in defs.items()))
            _run([NVCC, "-O3", "-std=c++17", "-fmad=false", "-gencode", "arch=compute_100a,code=compute_100a", "-ptx",
                  "-include", hdr, src, "-o", out], out + ".log")
            text = open(out).read()
            assert text.count("FXJIT_BODY ") == 1 and ')FXPTX"' not in text, out
            assert text.count("FXJIT_DEFORM ") == (1 if cplx else 0), out
            return text
        tjobs = [(False, nx, m) for nx in JIT_NX for m in range(4)] + [(True, n, m) for n in CPLX_DIMS for m in range(4)]
        with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
            texts = list(ex.map(ptx, tjobs))
        with open(tpl_inc, "w") as f:
            f.write("// GENERATED by build.py from fx_jit_template*.cu (nvcc -ptx) -- do not edit.\n")
            for (cplx, n, mode), t in zip(tjobs, texts):
                f.write('static const char fx_jit_template_ptx_%s%d_m%d[] = R"FXPTX(%s)FXPTX";\n'
                        % ("c" if cplx else "r", n, mode, t))
            f.write("static const char *fx_jit_template_lookup(bool cplx, int n, int mode) {\n")
            for (cplx, n, mode) in tjobs:
                f.write("  if (cplx == %s && n == %d && mode == %d) return fx_jit_template_ptx_%s%d_m%d;\n"
                        % ("true" if cplx else "false", n, mode, "c" if cplx else "r", n, mode))
            f.write("  return nullptr;\n}\n")
    jobs = []  # (object, cmd, sources)

    def cu(name, src, extra=()):
        o = os.path.join(OBJ, name + ".o")
        s = os.path.join(CSRC, src)
        jobs.append((o, [NVCC] + NVFLAGS + list(extra) + ["-c", s, "-o", o], [s] + hdrs))

    cu("fx_kernels_real", "fx_kernels_real.cu")
    cu("fx_kernels_small", "fx_kernels_small.cu")
    cu("fx_kernels_dd", "fx_kernels_dd.cu")
    cu("fx_kernels_cubature", "fx_kernels_cubature.cu")
    cu("fx_kernels_noalloc", "fx_kernels_noalloc.cu")
    for n in CPLX_DIMS:
        cu("fx_kernels_cplx_n%d" % n, "fx_kernels_cplx.cu", ["-DFX_N=%d" % n])
    for name in ("fiesta_abi", "fx_compiler", "fx_jit"):
        o = os.path.join(OBJ, name + ".o")
        s = os.path.join(CSRC, name + ".cpp")
        jobs.append((o, ["g++", "-O2", "-std=c++17", "-fPIC", "-pthread", "-DFXJ_P_VEGAS=%d" % P_VEGAS,
                         "-I/usr/local/cuda/include", "-c", s, "-o", o],
                     [s] + hdrs + ([tpl_inc] if name == "fx_jit" else [])))
    todo = [(o, c) for (o, c, srcs) in jobs if force or _stale(o, srcs)]
    if verbose and todo:
        print("building %d objects" % len(todo), file=sys.stderr)
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
        list(ex.map(lambda oc: _run(oc[1], oc[0] + ".log"), todo))
    objs = [o for (o, _, _) in jobs]
    if force or todo or _stale(LIB, objs):
        _run([NVCC, "-shared", "-o", LIB] + ARCH + objs + ["-lcudart", "-lnvptxcompiler_static", "-lpthread", "-ldl"], os.path.join(OBJ, "link.log"))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
