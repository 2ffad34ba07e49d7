#!/usr/bin/env python
"""Generates fx_interp_gen.inc: the fast path of the program walk as inline PTX.

Why PTX: nvcc lowers a C++ `switch` over ~400 opcodes to a compare-and-branch tree, and ptxas
then re-copies the whole per-thread register state (X, S, A: 140+ registers) on every trip
round the loop -- measured at ~600 cycles per interpreted op (profiles/r01_switch_baseline.md).
Here the dispatch is one `brx.idx` through a `.branchtargets` table (SASS: LDC from the jump table,
BRX), every handler names its operand registers statically and returns to the single dispatch
point, so the loop is: LDS (opcode, prefetched), LDS.64 (immediate), decode, LDC, BRX, P x DFMA, BRA.
Threaded code (a dispatch at the end of every handler) was measured twice and is slower on sm_100a
(ptxas gives every brx.idx site its own constant-bank table, or, without the
optimizer constant bank, its own island of BRA instructions).

One function per (arithmetic type, NX variables, P points per thread):

    fx_fast_<real|cplx>_<NX>_<P>(A, X, S, pc, mem, w0, w2, w3)

walks instructions from shared-memory byte address `pc` until it meets an opcode it does not
handle (FX_OUT, FX_END, log/exp, complex division ...), and returns that instruction's words in
(w0, w2, w3) with pc pointing past it; the C++ caller (fx_interp.cuh) handles it and re-enters.

    python gen_interp_ptx.py > fx_interp_gen.inc      (build.py does this)

The opcode numbers are parsed from fx_isa.h, so the two cannot drift apart.
"""
import os
import re
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
# threaded code (every handler ends with its own fetch + brx.idx) saves one BRA per op, but gives
# ptxas a control-flow graph of (#handlers x #opcodes) edges: its compile time explodes (> 30 min
# for NX = 8).  With one shared dispatch point the graph has #handlers + #opcodes edges.
THREADED = False
THREADS = 128   # FX_THREADS: stride (in doubles) between spill slots of one thread


def parse_isa():
    """opcode names -> numbers, evaluating the `= expr` forms of fx_isa.h with its #defines."""
    txt = open(os.path.join(HERE, "fx_isa.h")).read()
    env = {}
    for m in re.finditer(r"^#define\s+(FX_\w+)\s+(.+?)\s*(?://.*)?$", txt, re.M):
        name, val = m.group(1), m.group(2)
        if "(" in name:
            continue
        try:
            env[name] = int(eval(val, {}, env))
        except Exception:
            pass
    body = txt[txt.index("enum fx_op"):]
    body = body[body.index("{") + 1:body.index("};")]
    ops, val = {}, 0
    for line in body.splitlines():
        line = line.split("//")[0].strip().rstrip(",")
        if not line:
            continue
        m = re.match(r"(\w+)\s*=\s*(.+)$", line)
        if m:
            val = int(eval(m.group(2), {}, {**env, **ops}))
            ops[m.group(1)] = val
        else:
            ops[line] = val
        val += 1
    return ops, env


OPS, ENV = parse_isa()
NOPS = OPS["FX_NOPS"]
NXMAX, NS, NL, NR = ENV["FX_NXMAX"], ENV["FX_NS"], ENV["FX_L"], ENV["FX_NR"]


class Gen:
    def __init__(self, cplx, nx, p):
        self.cplx, self.nx, self.p = cplx, nx, p
        self.operands = []       # (constraint, c-expression)
        self.lines = []
        self.marks = []          # (first line index, label) of every handler
        self.C = 2 if cplx else 1

    # ---- operands ---------------------------------------------------------------------
    def opnd(self, constraint, expr):
        self.operands.append((constraint, expr))
        return "%%%d" % (len(self.operands) - 1)

    def setup(self):
        comp = (".re", ".im") if self.cplx else ("",)
        self.AL = [[[self.opnd("+d", f"A[{d}][{p}]{c}") for c in comp] for p in range(self.p)] for d in range(NL)]
        self.A = self.AL[0]
        self.X = [[[self.opnd("+d", f"X[{k}][{p}]{c}") for c in comp] for p in range(self.p)] for k in range(self.nx)]
        self.S = [[[self.opnd("+d", f"S[{j}][{p}]{c}") for c in comp] for p in range(self.p)] for j in range(NS)]
        self.pc = self.opnd("+r", "pc")
        self.w0 = self.opnd("=r", "w0")
        self.w2 = self.opnd("=r", "w2")
        self.w3 = self.opnd("=r", "w3")
        self.mem = self.opnd("r", "mem")

    def R(self, r):
        return self.X[r] if r < NXMAX else self.S[r - NXMAX]

    def emit(self, s):
        self.lines.append(s)

    def dispatch(self):
        """Fetch + decode + indirect branch.  Split fetch: the opcode word of op i+1 is loaded one op
        ahead (so decode -> table lookup -> BRX never waits on shared memory), the immediate of op i
        is loaded at dispatch and arrives while the branch resolves.  No register copies: an
        earlier version prefetched the whole 16-byte word and paid 8 MOVs per op for it."""
        self.emit("and.b32 op, nop, 0xffff;")
        self.emit(f"ld.shared.f64 imm, [{self.pc}+8];")
        self.emit(f"ld.shared.u32 nop, [{self.pc}+16];")
        self.emit(f"add.u32 {self.pc}, {self.pc}, 16;")
        self.emit("brx.idx.uni op, TBL;")

    # ---- memory slots -----------------------------------------------------------------
    def mem_addr(self):
        """ma = mem + aux * (C*P*THREADS*8)"""
        self.emit(f"ld.shared.u32 ma, [{self.pc}+-16];")
        self.emit("shr.u32 ma, ma, 16;")
        self.emit(f"mad.lo.u32 ma, ma, {self.C * self.p * THREADS * 8}, {self.mem};")

    def mem_off(self, p, c):
        return (c * self.p + p) * THREADS * 8

    def ld_mem(self, p):
        """loads slot value of point p into m0 (re) [, m1 (im)]"""
        for c in range(self.C):
            self.emit(f"ld.shared.f64 m{c}, [ma+{self.mem_off(p, c)}];")
        return ["m0", "m1"][:self.C]

    # ---- arithmetic templates; a, b, c are component lists; result assigned to a ------
    def fma_full(self, a, b, c):          # a = a*b + c
        if not self.cplx:
            self.emit(f"fma.rn.f64 {a[0]}, {a[0]}, {b[0]}, {c[0]};")
            return
        self.emit(f"neg.f64 t0, {a[1]};")
        self.emit(f"fma.rn.f64 t0, t0, {b[1]}, {c[0]};")
        self.emit(f"fma.rn.f64 t1, {a[1]}, {b[0]}, {c[1]};")
        self.emit(f"fma.rn.f64 t1, {a[0]}, {b[1]}, t1;")
        self.emit(f"fma.rn.f64 {a[0]}, {a[0]}, {b[0]}, t0;")
        self.emit(f"mov.f64 {a[1]}, t1;")

    def fma_c(self, a, b, imm="imm"):     # a = a*b + imm (imm real)
        if not self.cplx:
            self.emit(f"fma.rn.f64 {a[0]}, {a[0]}, {b[0]}, {imm};")
            return
        self.emit(f"neg.f64 t0, {a[1]};")
        self.emit(f"fma.rn.f64 t0, t0, {b[1]}, {imm};")
        self.emit(f"mul.rn.f64 t1, {a[1]}, {b[0]};")
        self.emit(f"fma.rn.f64 t1, {a[0]}, {b[1]}, t1;")
        self.emit(f"fma.rn.f64 {a[0]}, {a[0]}, {b[0]}, t0;")
        self.emit(f"mov.f64 {a[1]}, t1;")

    def fma_rc(self, a, r, imm="imm"):    # a = r*imm + a
        for c in range(self.C):
            self.emit(f"fma.rn.f64 {a[c]}, {r[c]}, {imm}, {a[c]};")

    def fma_up(self, a, u, r):            # a = u*r + a
        if not self.cplx:
            self.emit(f"fma.rn.f64 {a[0]}, {u[0]}, {r[0]}, {a[0]};")
            return
        self.emit(f"neg.f64 t0, {u[1]};")
        self.emit(f"fma.rn.f64 t0, t0, {r[1]}, {a[0]};")
        self.emit(f"fma.rn.f64 {a[0]}, {u[0]}, {r[0]}, t0;")
        self.emit(f"fma.rn.f64 t1, {u[1]}, {r[0]}, {a[1]};")
        self.emit(f"fma.rn.f64 {a[1]}, {u[0]}, {r[1]}, t1;")

    def mul(self, a, b):                  # a = a*b
        if not self.cplx:
            self.emit(f"mul.rn.f64 {a[0]}, {a[0]}, {b[0]};")
            return
        self.emit(f"mul.rn.f64 t0, {a[1]}, {b[1]};")
        self.emit("neg.f64 t0, t0;")
        self.emit(f"mul.rn.f64 t1, {a[1]}, {b[0]};")
        self.emit(f"fma.rn.f64 t1, {a[0]}, {b[1]}, t1;")
        self.emit(f"fma.rn.f64 {a[0]}, {a[0]}, {b[0]}, t0;")
        self.emit(f"mov.f64 {a[1]}, t1;")

    def comp2(self, ins, a, x, y):        # a = x <ins> y componentwise
        for c in range(self.C):
            self.emit(f"{ins} {a[c]}, {x[c]}, {y[c]};")

    # ---- handlers ---------------------------------------------------------------------
    def prio(self, label):
        """Layout order: the handlers sparse-polynomial programs live in come first and contiguous,
        so that their union stays inside the 32 KB L1.5 instruction cache (the first layout spread
        them over 87 KB: icc hit rate 60 %, 'no instruction' the top stall)."""
        m = re.match(r"H_([A-Z_]+?)(?:_(\d+))?(?:_(\d+))?$", label)
        fam = m.group(1)
        nums = [int(g) for g in m.groups()[1:] if g is not None]
        r = nums[-1] if len(nums) == 2 else None
        isx = r is not None and r < NXMAX
        if fam in ("MULC_R", "MUL_R", "FMA_AR_C", "FMA_RC_A", "FMA_UP") and isx:
            return 0
        if fam in ("LDC", "ADDC", "MULC", "ADD_UP", "MUL_UP", "FMA_UPC", "ST_S", "NEG", "SQR", "RSUBC"):
            return 1
        if "DIV" in fam or fam == "SQRT":
            return 9
        if fam.endswith("M") or "_AM_" in fam or "_MC_" in fam or fam == "FMA_AR_M":
            return 5
        return 2 if isx else 3

    def handler(self, label, body_per_point, pre=None):
        self.marks.append((len(self.lines), label))
        self.emit(f"{label}:")
        if pre:
            pre()
        for p in range(self.p):
            body_per_point(p)
        if THREADED:
            self.dispatch()
        else:
            self.emit("bra.uni NEXT;")

    def build(self):
        self.setup()
        table = ["EXIT"] * NOPS
        AL, cx, C = self.AL, self.cplx, self.C

        def regs():
            return [r for r in range(NR) if not (r < NXMAX and r >= self.nx)]

        def lr_family(name, body, pre=None, dmax=NL):
            """opcode = base + d*NR + r; body(a, r, d, p)"""
            for d in range(dmax):
                for r in regs():
                    lab = f"H_{name}_{d}_{r}"
                    table[OPS["FX_" + name] + d * NR + r] = lab
                    self.handler(lab, lambda p, d=d, r=r: body(AL[d][p], self.R(r)[p], d, p), pre)

        def l_family(name, body, pre=None, dmax=NL):
            """opcode = base + d; body(a, d, p)"""
            for d in range(dmax):
                lab = f"H_{name}_{d}"
                table[OPS["FX_" + name] + d] = lab
                self.handler(lab, lambda p, d=d: body(AL[d][p], d, p), pre)

        def r0_family(name, body, ok=True):
            if not ok:
                return
            for r in regs():
                lab = f"H_{name}_0_{r}"
                table[OPS["FX_" + name] + r] = lab
                self.handler(lab, lambda p, r=r: body(AL[0][p], self.R(r)[p], p))

        E = self.emit
        lr_family("MULC_R", lambda a, r, d, p: [E(f"mul.rn.f64 {a[c]}, {r[c]}, imm;") for c in range(C)])
        lr_family("MUL_R", lambda a, r, d, p: self.mul(a, r))
        lr_family("FMA_AR_C", lambda a, r, d, p: self.fma_c(a, r))
        lr_family("FMA_RC_A", lambda a, r, d, p: self.fma_rc(a, r))
        lr_family("FMA_UP", lambda a, r, d, p: self.fma_up(a, AL[d + 1][p], r), dmax=NL - 1)
        lr_family("ADD_R", lambda a, r, d, p: self.comp2("add.rn.f64", a, a, r))
        lr_family("LD_R", lambda a, r, d, p: [E(f"mov.f64 {a[c]}, {r[c]};") for c in range(C)])
        lr_family("FMA_AR_M", lambda a, r, d, p: self.fma_full(a, r, self.ld_mem(p)), pre=self.mem_addr)

        def ldc(a, d, p):
            E(f"mov.f64 {a[0]}, imm;")
            if cx:
                E(f"mov.f64 {a[1]}, zero;")

        l_family("LDC", ldc)
        l_family("ADDC", lambda a, d, p: E(f"add.rn.f64 {a[0]}, {a[0]}, imm;"))
        l_family("MULC", lambda a, d, p: [E(f"mul.rn.f64 {a[c]}, {a[c]}, imm;") for c in range(C)])
        l_family("ADD_UP", lambda a, d, p: self.comp2("add.rn.f64", a, a, AL[d + 1][p]), dmax=NL - 1)
        l_family("MUL_UP", lambda a, d, p: self.mul(a, AL[d + 1][p]), dmax=NL - 1)
        l_family("LDM", lambda a, d, p: [E(f"mov.f64 {a[c]}, {m};") for c, m in enumerate(self.ld_mem(p))], self.mem_addr)
        l_family("STM", lambda a, d, p: [E(f"st.shared.f64 [ma+{self.mem_off(p, c)}], {a[c]};") for c in range(C)],
                 self.mem_addr)
        l_family("ADDM", lambda a, d, p: self.comp2("add.rn.f64", a, a, self.ld_mem(p)), self.mem_addr)
        l_family("MULM", lambda a, d, p: self.mul(a, self.ld_mem(p)), self.mem_addr)
        l_family("FMA_MC_A", lambda a, d, p: self.fma_rc(a, self.ld_mem(p)), self.mem_addr)
        l_family("FMA_AM_C", lambda a, d, p: self.fma_c(a, self.ld_mem(p)), self.mem_addr)
        l_family("FMA_UPC", lambda a, d, p: self.fma_rc(a, AL[d + 1][p]), dmax=NL - 1)

        r0_family("SUB_R", lambda a, r, p: self.comp2("sub.rn.f64", a, a, r))
        r0_family("RSUB_R", lambda a, r, p: self.comp2("sub.rn.f64", a, r, a))
        r0_family("DIV_R", lambda a, r, p: E(f"div.rn.f64 {a[0]}, {a[0]}, {r[0]};"), ok=not cx)
        r0_family("RDIV_R", lambda a, r, p: E(f"div.rn.f64 {a[0]}, {r[0]}, {a[0]};"), ok=not cx)
        A = AL[0]
        for j in range(NS):
            lab = f"H_ST_S_{j}"
            table[OPS["FX_ST_S"] + j] = lab
            self.handler(lab, lambda p, j=j: [E(f"mov.f64 {self.S[j][p][c]}, {A[p][c]};") for c in range(C)])

        def single(name, body, pre=None, ok=True):
            if not ok:
                return
            lab = "H_" + name
            table[OPS["FX_" + name]] = lab
            self.handler(lab, body, pre)

        def rsubc(p):
            E(f"sub.rn.f64 {A[p][0]}, imm, {A[p][0]};")
            if cx:
                E(f"neg.f64 {A[p][1]}, {A[p][1]};")

        single("RSUBC", rsubc)
        single("DIVC", lambda p: [E(f"div.rn.f64 {A[p][c]}, {A[p][c]}, imm;") for c in range(C)])
        single("RDIVC", lambda p: E(f"div.rn.f64 {A[p][0]}, imm, {A[p][0]};"), ok=not cx)
        single("SUBM", lambda p: self.comp2("sub.rn.f64", A[p], A[p], self.ld_mem(p)), self.mem_addr)
        single("RSUBM", lambda p: self.comp2("sub.rn.f64", A[p], self.ld_mem(p), A[p]), self.mem_addr)
        single("DIVM", lambda p: E(f"div.rn.f64 {A[p][0]}, {A[p][0]}, {self.ld_mem(p)[0]};"), self.mem_addr, ok=not cx)
        single("RDIVM", lambda p: E(f"div.rn.f64 {A[p][0]}, {self.ld_mem(p)[0]}, {A[p][0]};"), self.mem_addr, ok=not cx)
        single("NEG", lambda p: [E(f"neg.f64 {A[p][c]}, {A[p][c]};") for c in range(C)])
        single("SQR", lambda p: self.mul(A[p], A[p]))
        single("SQRT", lambda p: E(f"sqrt.rn.f64 {A[p][0]}, {A[p][0]};"), ok=not cx)
        return table

    def function(self):
        table = self.build()
        ends = [m[0] for m in self.marks[1:]] + [len(self.lines)]
        blocks = [(self.prio(lab), i, self.lines[a:b]) for i, ((a, lab), b) in enumerate(zip(self.marks, ends))]
        handlers = [ln for _, _, blk in sorted(blocks, key=lambda t: (t[0], t[1])) for ln in blk]
        self.lines = []
        kind = "cplx" if self.cplx else "real"
        T = "cplx" if self.cplx else "double"
        name = f"fx_fast_{kind}_{self.nx}_{self.p}"
        out = [f"#if FX_WANT({int(self.cplx)}, {self.nx}, {self.p})",
               f"__device__ __forceinline__ void {name}({T} (&A)[{NL}][{self.p}], {T} (&X)[{self.nx}][{self.p}], "
               f"{T} (&S)[{NS}][{self.p}], uint32_t &pc, uint32_t mem, uint32_t &w0, uint32_t &w2, uint32_t &w3) {{",
               "  asm volatile(", '    "{\\n"',
               '    ".reg .u32 nop, op, ma;\\n"', '    ".reg .f64 imm, zero, t0, t1, m0, m1;\\n"',
               '    "mov.f64 zero, 0d0000000000000000;\\n"']
        tl = ", ".join(table)
        out.append(f'    "TBL: .branchtargets {tl};\\n"')
        self.emit(f"ld.shared.u32 nop, [{self.pc}];")
        self.emit("NEXT:")
        self.dispatch()
        for ln in self.lines + handlers:
            out.append(f'    "{ln}\\n"')
        out.append('    "EXIT:\\n"')
        out.append(f'    "ld.shared.u32 {self.w0}, [{self.pc}+-16];\\n"')
        out.append(f'    "mov.b64 {{{self.w2},{self.w3}}}, imm;\\n"')
        out.append('    "}\\n"')
        outs = [o for o in self.operands if o[0][0] in "+="]
        ins = [o for o in self.operands if o[0][0] not in "+="]
        # outputs must be numbered first: check the numbering matches the order used above
        order = outs + ins
        assert order == self.operands, "operand order must be outputs then inputs"
        out.append("    : " + ", ".join(f'"{c}"({e})' for c, e in outs))
        out.append("    : " + ", ".join(f'"{c}"({e})' for c, e in ins))
        out.append('    : "memory");')
        out.append("}")
        out.append(f"template <> struct fx_fast<{T}, {self.nx}, {self.p}> {{")
        out.append(f"  static __device__ __forceinline__ void run({T} (&A)[{NL}][{self.p}], {T} (&X)[{self.nx}][{self.p}], "
                   f"{T} (&S)[{NS}][{self.p}], uint32_t &pc, uint32_t mem, uint32_t &w0, uint32_t &w2, uint32_t &w3) {{")
        out.append(f"    {name}(A, X, S, pc, mem, w0, w2, w3);")
        out.append("  }")
        out.append("};")
        out.append("#endif")
        return "\n".join(out)


def main():
    variants = [(False, nx, 4) for nx in (4, 8, 12)] + [(False, nx, 1) for nx in range(1, 9)] + \
               [(True, nx, 1) for nx in range(1, 9)]
    print("// GENERATED by gen_interp_ptx.py -- do not edit.  See that file for the design.")
    for cplx, nx, p in variants:
        print(Gen(cplx, nx, p).function())


if __name__ == "__main__":
    main()
