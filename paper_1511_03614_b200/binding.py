"""ctypes binding of include/fiesta_b200.h -- same names, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libfiesta_b200.so")

RULE_LATTICE, RULE_MC, RULE_VEGAS = 0, 1, 2
MODE_EVAL, N_MODES = 3, 4
TIER_ANY, TIER_INTERPRETER, TIER_NATIVE = -1, 0, 1
MAX_ORDERS = 8

RESULT_DTYPE = np.dtype([("re", "f8"), ("re_err", "f8"), ("im", "f8"), ("im_err", "f8"), ("chi2", "f8"),
                         ("neval", "u8"), ("n_nonfinite", "u8")])
INFO_DTYPE = np.dtype([("n_ir_ops", "i4"), ("n_fp64_ops", "i4"), ("n_fma", "i4"), ("n_log", "i4"), ("n_exp", "i4"),
                       ("n_div", "i4"), ("n_reg_temps", "i4"), ("n_mem_slots", "i4"), ("n_deform_ops", "i4"),
                       ("flops", "f8")], align=True)

E_NONFINITE = -6
ERROR_NAMES = {-1: "FIESTA_E_PARSE", -2: "FIESTA_E_DIM", -3: "FIESTA_E_NOTPOLY", -4: "FIESTA_E_RULE",
               -5: "FIESTA_E_CUDA", -6: "FIESTA_E_NONFINITE", -7: "FIESTA_E_ARG", -8: "FIESTA_E_TOOBIG"}


class FiestaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERROR_NAMES.get(code, code)}: {msg}")
        self.code = code


class _SectorDesc(C.Structure):
    _fields_ = [("sector_id", C.c_int32), ("n_orders", C.c_int32), ("expr", C.POINTER(C.c_char_p)),
                ("is_complex", C.c_int32), ("deform_f_index", C.c_int32), ("lam", C.c_double)]


class _TestF(C.Structure):
    _fields_ = [("n_points", C.c_uint64), ("n_bad", C.c_uint64), ("max_im_f", C.c_double), ("min_abs_f", C.c_double),
                ("lam", C.c_double)]


class _Rule(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_shifts", C.c_int32), ("korobov_a", C.c_uint64),
                ("genvec", C.POINTER(C.c_uint64)), ("periodize_r", C.c_int32), ("vegas_bins", C.c_int32),
                ("vegas_iters", C.c_int32), ("vegas_alpha", C.c_double)]


_VP = C.c_void_p
_I32 = C.c_int32
_U64 = C.c_uint64
_SIGNATURES = {
    "fiesta_create": (C.c_int, [C.POINTER(_VP), C.c_int, _VP]),
    "fiesta_destroy": (None, [_VP]),
    "fiesta_last_error": (C.c_char_p, [_VP]),
    "fiesta_compile": (C.c_int, [_VP, C.POINTER(_SectorDesc), _I32, _I32, C.POINTER(_VP), _VP]),
    "fiesta_program_free": (None, [_VP]),
    "fiesta_integrate": (C.c_int, [_VP, _VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, _VP]),
    "fiesta_integrate_async": (C.c_int, [_VP, _VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64]),
    "fiesta_fetch_results": (C.c_int, [_VP, _I32, _I32, _VP]),
    "fiesta_last_timing": (C.c_int, [_VP, C.POINTER(C.c_double), C.POINTER(_I32)]),
    "fiesta_eval_points": (C.c_int, [_VP, _VP, _I32, _VP, _U64, _VP]),
    "fiesta_generate_points": (C.c_int, [_VP, C.POINTER(_Rule), _U64, _I32, _I32, _U64, _U64, _U64, _I32, _VP]),
    "fiesta_transform_points": (C.c_int, [_VP, C.POINTER(_Rule), _VP, _U64, _I32, _VP, _VP, _VP]),
    "fiesta_partial_sums": (C.c_int, [_VP, _VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, _VP]),
    "fiesta_vegas_iteration": (C.c_int, [_VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, _I32, _VP, _VP, _VP]),
    "fiesta_vegas_refine": (C.c_int, [_VP, _I32, _I32, C.c_double, _VP, _VP, _VP]),
    "fiesta_vegas_grid": (C.c_int, [_VP, _I32, _I32, _I32, _VP, _VP]),
    "fiesta_combine": (C.c_int, [_VP, _I32, _I32, _VP]),
    "fiesta_program_dump": (C.c_int, [_VP, _I32, C.c_char_p, _U64]),
    "fiesta_program_native": (C.c_int, [_VP, _I32, _I32, C.c_char_p, _U64]),
    "fiesta_program_wait_native": (C.c_int, [_VP, _I32, C.c_double]),
    "fiesta_program_native_stats": (C.c_int, [_VP, C.POINTER(_I32), C.POINTER(_I32), C.POINTER(C.c_double), C.POINTER(_I32)]),
    "fiesta_native_assemble": (C.c_int, [_VP, _I32, _I32, C.c_char_p, _U64, C.POINTER(_U64), C.c_char_p, _U64]),
    "fiesta_integrate_tier": (C.c_int, [_VP, _VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, _I32, _VP]),
    "fiesta_last_tiers": (C.c_int, [_VP, C.POINTER(_I32), C.POINTER(_I32)]),
    "fiesta_eval_points_tier": (C.c_int, [_VP, _VP, _I32, _I32, _VP, _U64, _VP]),
    "fiesta_partial_sums_tier": (C.c_int, [_VP, _VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, _I32, _VP]),
    "fiesta_chunk_sums": (C.c_int, [_VP, _VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, _I32, C.POINTER(_U64),
                                    C.POINTER(_I32), _VP]),
    "fiesta_vegas_iteration_tier": (C.c_int, [_VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, _I32, _I32, _VP, _VP,
                                              _VP]),
    "fiesta_fp64_peak": (C.c_int, [_VP, C.c_double, C.POINTER(C.c_double)]),
    "fiesta_test_f": (C.c_int, [_VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, C.c_double, C.POINTER(_TestF)]),
    "fiesta_select_lambda": (C.c_int, [_VP, _VP, _I32, _I32, _U64, _U64, C.c_double, _I32, _I32, C.POINTER(C.c_double),
                                       C.POINTER(_TestF)]),
    "fiesta_program_set_lambda": (C.c_int, [_VP, _VP, _I32, C.c_double]),
    "fiesta_integrate_cubature": (C.c_int, [_VP, _VP, _VP, _I32, C.c_double, C.c_double, _U64, _I32, _VP, _VP]),
    "fiesta_cubature_rule": (C.c_int, [_VP, _VP, _I32, _I32, _VP, _U64, _VP, _VP, _VP, _VP]),
    "fiesta_partial_sums_shifts": (C.c_int, [_VP, _VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, _I32, _I32, _I32, _VP]),
    "fiesta_last_nonfinite": (C.c_int, [_VP, _I32, _VP]),
    "fiesta_estimate_from_sums": (C.c_int, [_VP, _VP, _VP, _I32, _I32, _U64, _VP, _VP, _VP]),
    "fiesta_partial_sums_noalloc_async": (C.c_int, [_VP, _VP, _I32, _I32, _U64, C.POINTER(_Rule), _U64, _VP, _VP]),
    "fiesta_set_mixed": (C.c_int, [_VP, C.c_double]),
    "fiesta_eval_points_dd": (C.c_int, [_VP, _VP, _I32, _VP, _U64, _VP]),
}

_lib = None


def exported_symbols():
    """Names include/fiesta_b200.h declares (the binding covers every one)."""
    return sorted(_SIGNATURES)


def load_library():
    """dlopen libfiesta_b200.so (fails loudly if it has not been built) and set the prototypes."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1511_03614_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


@dataclass
class Rule:
    """Mirror of `fiesta_rule`."""
    kind: int = RULE_LATTICE
    n_shifts: int = 1
    korobov_a: int = 1
    genvec: object = None          # optional sequence of dim integers
    periodize_r: int = 3
    vegas_bins: int = 50
    vegas_iters: int = 10
    vegas_alpha: float = 1.5

    @classmethod
    def from_workload(cls, wl):
        return cls(kind=wl.rule, n_shifts=wl.n_shifts, korobov_a=wl.korobov_a, periodize_r=wl.periodize_r,
                   vegas_bins=wl.vegas_bins, vegas_iters=wl.vegas_iters, vegas_alpha=wl.vegas_alpha)

    def _c(self):
        r = _Rule(self.kind, self.n_shifts, self.korobov_a, None, self.periodize_r, self.vegas_bins,
                  self.vegas_iters, self.vegas_alpha)
        keep = None
        if self.genvec is not None:
            keep = (C.c_uint64 * len(self.genvec))(*[int(g) for g in self.genvec])
            r.genvec = C.cast(keep, C.POINTER(C.c_uint64))
        return r, keep


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_VP)


def native_assemble(sector, dim, mode=RULE_LATTICE, buflen=1 << 23):
    """fiesta_native_assemble: host only.  sector: object with .sector_id, .texts (workloads.SectorText).
    -> (generated PTX of the program body/bodies, bytes of the assembled sm_100a cubin, the assembler's
    resource report)."""
    lib = load_library()
    arr = (C.c_char_p * len(sector.texts))(*[t.encode() for t in sector.texts])
    d = _SectorDesc(int(sector.sector_id), len(sector.texts), C.cast(arr, C.POINTER(C.c_char_p)),
                    int(bool(sector.is_complex)), int(sector.deform_f_index), float(sector.lam))
    buf = C.create_string_buffer(buflen)
    info = C.create_string_buffer(1 << 14)
    n = _U64(0)
    rc = lib.fiesta_native_assemble(C.byref(d), int(dim), int(mode), buf, buflen, C.byref(n), info, 1 << 14)
    if rc != 0:
        raise FiestaError(rc, buf.value.decode(errors="replace"))
    return buf.value.decode(), int(n.value), info.value.decode(errors="replace")


class Program:
    """Handle of a compiled `fiesta_program` (owned; freed on close / garbage collection)."""

    def __init__(self, ctx, handle, nsectors, dim, K, is_complex, info):
        self.ctx, self.handle, self.nsectors, self.dim = ctx, handle, nsectors, dim
        self.K, self.is_complex, self.info = K, is_complex, info

    def close(self):
        if self.handle:
            load_library().fiesta_program_free(self.handle)
            self.handle = None

    __del__ = close

    def native(self, sector=0, mode=RULE_LATTICE):
        """(the native kernel of (sector, mode) is ready, the assembler's report or the reason if not)
        -- fiesta_program_native"""
        buf = C.create_string_buffer(1 << 14)
        rc = load_library().fiesta_program_native(self.handle, sector, mode, buf, 1 << 14)
        if rc < 0:
            raise FiestaError(rc, "fiesta_program_native")
        return bool(rc), buf.value.decode(errors="replace")

    def wait_native(self, mode=RULE_LATTICE, timeout_s=-1.0):
        """Request the `mode` kernels of all sectors and wait for the background assembly; -> number ready."""
        rc = load_library().fiesta_program_wait_native(self.handle, int(mode), float(timeout_s))
        if rc < 0:
            raise FiestaError(rc, "fiesta_program_wait_native")
        return rc

    def native_stats(self):
        """-> dict(assembled, cache_hits, cpu_seconds, threads) of the background assembly so far."""
        a, h, t, n = _I32(), _I32(), C.c_double(), _I32()
        load_library().fiesta_program_native_stats(self.handle, C.byref(a), C.byref(h), C.byref(t), C.byref(n))
        return dict(assembled=a.value, cache_hits=h.value, cpu_seconds=t.value, threads=n.value)

    def dump(self, sector=0, buflen=1 << 20):
        buf = C.create_string_buffer(buflen)
        self.ctx._check(load_library().fiesta_program_dump(self.handle, sector, buf, buflen))
        return buf.value.decode()


class Context:
    """Handle of a `fiesta_ctx` bound to one CUDA device and stream (a raw cudaStream_t integer,
    e.g. `torch.cuda.current_stream().cuda_stream`; 0 = default stream)."""

    def __init__(self, device=0, stream=0):
        self.lib = load_library()
        h = _VP()
        rc = self.lib.fiesta_create(C.byref(h), int(device), _VP(int(stream)))
        if rc:
            raise FiestaError(rc, "fiesta_create failed (no sm_100 device? there is no CPU fallback)")
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            self.lib.fiesta_destroy(self.handle)
            self.handle = None

    __del__ = close

    def _check(self, rc, allow_nonfinite=False):
        if rc and not (allow_nonfinite and rc == E_NONFINITE):
            msg = self.lib.fiesta_last_error(self.handle)
            raise FiestaError(rc, msg.decode() if msg else "")
        return rc

    # ---- fiesta_compile ------------------------------------------------------------------
    def compile(self, sectors, dim):
        """sectors: objects with .sector_id, .texts (K strings), .is_complex, .deform_f_index, .lam
        (workloads.SectorText).  Returns a Program; .info is a numpy record array [nsectors]."""
        n = len(sectors)
        descs = (_SectorDesc * n)()
        keep = []
        for i, s in enumerate(sectors):
            arr = (C.c_char_p * len(s.texts))(*[t.encode() for t in s.texts])
            keep.append(arr)
            descs[i] = _SectorDesc(int(s.sector_id), len(s.texts), C.cast(arr, C.POINTER(C.c_char_p)),
                                   int(bool(s.is_complex)), int(s.deform_f_index), float(s.lam))
        info = np.zeros(n, dtype=INFO_DTYPE)
        assert INFO_DTYPE.itemsize == 48
        h = _VP()
        self._check(self.lib.fiesta_compile(self.handle, descs, n, int(dim), C.byref(h), _ptr(info)))
        return Program(self, h, n, int(dim), [len(s.texts) for s in sectors],
                       [bool(s.is_complex) or s.deform_f_index > 0 for s in sectors], info)

    # ---- fiesta_integrate ----------------------------------------------------------------
    def _sel(self, prog, sectors):
        if sectors is None:
            return None, prog.nsectors, list(range(prog.nsectors))
        a = np.ascontiguousarray(sectors, dtype=np.int32)
        return a, len(a), [int(i) for i in a]

    def integrate(self, prog, npoints, rule, seed, sectors=None, allow_nonfinite=False, tier=None):
        """-> numpy record array [nsectors][K] of RESULT_DTYPE.  tier: None (fiesta_integrate: whichever form
        of each sector is ready) or TIER_INTERPRETER / TIER_NATIVE (fiesta_integrate_tier)."""
        sel, nsel, idx = self._sel(prog, sectors)
        K = prog.K[idx[0]]
        out = np.zeros((nsel, K), dtype=RESULT_DTYPE)
        r, keep = rule._c()
        if tier is None:
            rc = self.lib.fiesta_integrate(self.handle, prog.handle, _ptr(sel), nsel, prog.dim, int(npoints),
                                           C.byref(r), int(seed), _ptr(out))
        else:
            rc = self.lib.fiesta_integrate_tier(self.handle, prog.handle, _ptr(sel), nsel, prog.dim, int(npoints),
                                                C.byref(r), int(seed), int(tier), _ptr(out))
        self._check(rc, allow_nonfinite)
        return out

    def last_tiers(self):
        """(sector passes of the last call served by a native kernel, by the interpreter)"""
        a, b = _I32(), _I32()
        self._check(self.lib.fiesta_last_tiers(self.handle, C.byref(a), C.byref(b)))
        return a.value, b.value

    def integrate_async(self, prog, npoints, rule, seed, sectors=None):
        sel, nsel, _ = self._sel(prog, sectors)
        r, keep = rule._c()
        self._check(self.lib.fiesta_integrate_async(self.handle, prog.handle, _ptr(sel), nsel, prog.dim,
                                                    int(npoints), C.byref(r), int(seed)))

    def fetch_results(self, nsectors, K, allow_nonfinite=False):
        out = np.zeros((nsectors, K), dtype=RESULT_DTYPE)
        self._check(self.lib.fiesta_fetch_results(self.handle, nsectors, K, _ptr(out)), allow_nonfinite)
        return out

    def last_timing(self):
        ms, n = C.c_double(), _I32()
        self._check(self.lib.fiesta_last_timing(self.handle, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    # ---- parity hooks --------------------------------------------------------------------
    def eval_points(self, prog, sector, x, tier=None):
        """x [npts][dim] float64 -> complex128 [npts][K] (weight excluded)."""
        x = np.ascontiguousarray(x, dtype=np.float64).reshape(-1, prog.dim)
        K = prog.K[sector]
        out = np.zeros((x.shape[0], K, 2), dtype=np.float64)
        if tier is None:
            rc = self.lib.fiesta_eval_points(self.handle, prog.handle, int(sector), _ptr(x), x.shape[0], _ptr(out))
        else:
            rc = self.lib.fiesta_eval_points_tier(self.handle, prog.handle, int(sector), int(tier), _ptr(x), x.shape[0],
                                                  _ptr(out))
        self._check(rc)
        return out[..., 0] + 1j * out[..., 1]

    def integrate_cubature(self, prog, epsrel=1e-6, epsabs=0.0, maxeval=1 << 22, sectors=None, tier=TIER_ANY,
                           allow_nonfinite=False):
        """Deterministic adaptive cubature -> (record array [nsectors][K] of RESULT_DTYPE, boxes per sector)."""
        sel, nsel, idx = self._sel(prog, sectors)
        out = np.zeros((nsel, prog.K[idx[0]]), dtype=RESULT_DTYPE)
        nboxes = np.zeros(nsel, dtype=np.uint64)
        self._check(self.lib.fiesta_integrate_cubature(self.handle, prog.handle, _ptr(sel), nsel, float(epsrel), float(epsabs),
                                                       int(maxeval), int(tier), _ptr(out), _ptr(nboxes)), allow_nonfinite)
        return out, nboxes

    def cubature_rule(self, prog, sector, boxes, tier=TIER_ANY):
        """boxes [nb][2][dim] (centre, half-widths) -> I7, I5 complex [nb][K], fourth differences [nb][dim], axis [nb]."""
        boxes = np.ascontiguousarray(boxes, dtype=np.float64).reshape(-1, 2, prog.dim)
        nb, K = boxes.shape[0], prog.K[int(sector)]
        i7, i5 = np.zeros((nb, K, 2)), np.zeros((nb, K, 2))
        fourth, axis = np.zeros((nb, prog.dim)), np.zeros(nb, dtype=np.int32)
        self._check(self.lib.fiesta_cubature_rule(self.handle, prog.handle, int(sector), int(tier), _ptr(boxes), nb, _ptr(i7),
                                                  _ptr(i5), _ptr(fourth), _ptr(axis)))
        return i7[..., 0] + 1j * i7[..., 1], i5[..., 0] + 1j * i5[..., 1], fourth, axis

    def partial_sums_noalloc_async(self, prog, sector, npoints, rule, seed, sums_dev, nonfinite_dev=0):
        """fiesta_partial_sums_noalloc_async: sums_dev / nonfinite_dev are raw DEVICE addresses (integers, e.g.
        tensor.data_ptr()) of [R][K][2] doubles and one uint64; queued on the context's stream, no synchronisation."""
        r, keep = rule._c()
        self._check(self.lib.fiesta_partial_sums_noalloc_async(self.handle, prog.handle, int(sector), prog.dim, int(npoints),
                                                               C.byref(r), int(seed), _VP(int(sums_dev)),
                                                               _VP(int(nonfinite_dev)) if nonfinite_dev else None))

    def set_mixed(self, small_x):
        """Mixed precision: points with min_k x_k < small_x are evaluated in double-double (0: off)."""
        self._check(self.lib.fiesta_set_mixed(self.handle, float(small_x)))

    def eval_points_dd(self, prog, sector, x):
        """Double-double walk of a real sector -> (hi, lo), each float64 [npts][K]."""
        x = np.ascontiguousarray(x, dtype=np.float64)
        out = np.zeros((x.shape[0], prog.K[int(sector)], 2))
        self._check(self.lib.fiesta_eval_points_dd(self.handle, prog.handle, int(sector), _ptr(x), x.shape[0], _ptr(out)))
        return out[..., 0], out[..., 1]

    def generate_points(self, rule, seed, sector_id, shift_or_iter, n_lattice, first, count, dim):
        t = np.zeros((count, dim), dtype=np.uint64)
        r, keep = rule._c()
        self._check(self.lib.fiesta_generate_points(self.handle, C.byref(r), int(seed), int(sector_id),
                                                    int(shift_or_iter), int(n_lattice), int(first), int(count),
                                                    int(dim), _ptr(t)))
        return t

    def transform_points(self, rule, t):
        t = np.ascontiguousarray(t, dtype=np.uint64)
        count, dim = t.shape
        x, xbar, w = np.zeros((count, dim)), np.zeros((count, dim)), np.zeros(count)
        r, keep = rule._c()
        self._check(self.lib.fiesta_transform_points(self.handle, C.byref(r), _ptr(t), count, dim, _ptr(x),
                                                     _ptr(xbar), _ptr(w)))
        return x, xbar, w

    def partial_sums(self, prog, npoints, rule, seed, sectors=None, tier=TIER_ANY):
        """-> float64 [nsectors][R][K][C][2] (S1, S2); all selected sectors must share K and C."""
        sel, nsel, idx = self._sel(prog, sectors)
        K, cc = prog.K[idx[0]], 2 if prog.is_complex[idx[0]] else 1
        R = rule.n_shifts if rule.kind == RULE_LATTICE else 1
        out = np.zeros((nsel, R, K, cc, 2), dtype=np.float64)
        r, keep = rule._c()
        self._check(self.lib.fiesta_partial_sums_tier(self.handle, prog.handle, _ptr(sel), nsel, prog.dim, int(npoints),
                                                      C.byref(r), int(seed), int(tier), _ptr(out)))
        return out

    def partial_sums_shifts(self, prog, npoints, rule, seed, shift_first, shift_count, sectors=None, tier=TIER_ANY):
        """The rows shift_first .. shift_first + shift_count - 1 of partial_sums -> ([nsectors][count][K][C][2],
        per-sector non-finite counts)."""
        sel, nsel, idx = self._sel(prog, sectors)
        K, cc = prog.K[idx[0]], 2 if prog.is_complex[idx[0]] else 1
        out = np.zeros((nsel, int(shift_count), K, cc, 2), dtype=np.float64)
        r, keep = rule._c()
        self._check(self.lib.fiesta_partial_sums_shifts(self.handle, prog.handle, _ptr(sel), nsel, prog.dim, int(npoints),
                                                        C.byref(r), int(seed), int(tier), int(shift_first), int(shift_count),
                                                        _ptr(out)))
        nf = np.zeros(nsel, dtype=np.uint64)
        self._check(self.lib.fiesta_last_nonfinite(self.handle, nsel, _ptr(nf)))
        return out, nf

    def estimate_from_sums(self, prog, sums, n_per_shift, nonfinite=None, sectors=None, allow_nonfinite=False):
        """sums [nsectors][R][K][C][2] -> record array [nsectors][K] (the estimator of fiesta_integrate, on the device)."""
        sel, nsel, idx = self._sel(prog, sectors)
        sums = np.ascontiguousarray(sums, dtype=np.float64)
        R = sums.shape[1]
        out = np.zeros((nsel, prog.K[idx[0]]), dtype=RESULT_DTYPE)
        nf = None if nonfinite is None else np.ascontiguousarray(nonfinite, dtype=np.uint64)
        self._check(self.lib.fiesta_estimate_from_sums(self.handle, prog.handle, _ptr(sel), nsel, R, int(n_per_shift), _ptr(sums),
                                                       _ptr(nf), _ptr(out)), allow_nonfinite)
        return out

    def chunk_sums(self, prog, npoints, rule, seed, sectors=None, tier=TIER_ANY):
        """-> (chunk_points, float64 [nsectors][R][nchunks][K][C][2]): every block's partial record."""
        sel, nsel, idx = self._sel(prog, sectors)
        K, cc = prog.K[idx[0]], 2 if prog.is_complex[idx[0]] else 1
        R = rule.n_shifts if rule.kind == RULE_LATTICE else 1
        r, keep = rule._c()
        cp, nch = _U64(), _I32()
        args = (self.handle, prog.handle, _ptr(sel), nsel, prog.dim, int(npoints), C.byref(r), int(seed), int(tier),
                C.byref(cp), C.byref(nch))
        self._check(self.lib.fiesta_chunk_sums(*args, None))
        out = np.zeros((nsel, R, nch.value, K, cc, 2), dtype=np.float64)
        self._check(self.lib.fiesta_chunk_sums(*args, _ptr(out)))
        return int(cp.value), out

    def vegas_iteration(self, prog, sector, npoints, rule, seed, iteration, grid, tier=TIER_ANY):
        grid = np.ascontiguousarray(grid, dtype=np.float64)
        K, cc = prog.K[sector], 2 if prog.is_complex[sector] else 1
        sums = np.zeros((K, cc, 2))
        hist = np.zeros((prog.dim, rule.vegas_bins))
        r, keep = rule._c()
        self._check(self.lib.fiesta_vegas_iteration_tier(self.handle, prog.handle, int(sector), prog.dim, int(npoints),
                                                         C.byref(r), int(seed), int(iteration), int(tier), _ptr(grid),
                                                         _ptr(sums), _ptr(hist)))
        return sums, hist

    def vegas_refine(self, grid, hist, alpha):
        grid = np.ascontiguousarray(grid, dtype=np.float64)
        hist = np.ascontiguousarray(hist, dtype=np.float64)
        nb = hist.shape[-1]
        ng = hist.size // nb
        out = np.zeros_like(grid)
        self._check(self.lib.fiesta_vegas_refine(self.handle, ng, nb, float(alpha), _ptr(grid), _ptr(hist), _ptr(out)))
        return out

    def vegas_grid(self, sector, dim, nbins):
        grid, hist = np.zeros((dim, nbins + 1)), np.zeros((dim, nbins))
        self._check(self.lib.fiesta_vegas_grid(self.handle, int(sector), dim, nbins, _ptr(grid), _ptr(hist)))
        return grid, hist

    def combine(self, per_sector):
        per_sector = np.ascontiguousarray(per_sector, dtype=RESULT_DTYPE)
        S, K = per_sector.shape
        tot = np.zeros(K, dtype=RESULT_DTYPE)
        self._check(self.lib.fiesta_combine(_ptr(per_sector), S, K, _ptr(tot)))
        return tot

    @staticmethod
    def _testf_dict(t):
        return dict(n_points=int(t.n_points), n_bad=int(t.n_bad), max_im_f=float(t.max_im_f), min_abs_f=float(t.min_abs_f),
                    lam=float(t.lam))

    def test_f(self, prog, sector, npoints, rule, seed, lam=-1.0):
        """fiesta_test_f -> dict(n_points, n_bad, max_im_f, min_abs_f, lam)."""
        r, keep = rule._c()
        out = _TestF()
        self._check(self.lib.fiesta_test_f(self.handle, prog.handle, int(sector), prog.dim, int(npoints), C.byref(r),
                                           int(seed), float(lam), C.byref(out)))
        return self._testf_dict(out)

    def select_lambda(self, prog, sector, npoints, seed, lambda_max=1.0, lambda_split=4, conservative=False):
        """fiesta_select_lambda -> (lambda, [test result of every candidate])."""
        lam = C.c_double()
        scan = (_TestF * int(lambda_split))()
        self._check(self.lib.fiesta_select_lambda(self.handle, prog.handle, int(sector), prog.dim, int(npoints), int(seed),
                                                  float(lambda_max), int(lambda_split), int(bool(conservative)),
                                                  C.byref(lam), scan))
        return lam.value, [self._testf_dict(t) for t in scan]

    def set_lambda(self, prog, sector, lam):
        self._check(self.lib.fiesta_program_set_lambda(self.handle, prog.handle, int(sector), float(lam)))

    def fp64_peak(self, ms_target=200.0):
        t = C.c_double()
        self._check(self.lib.fiesta_fp64_peak(self.handle, float(ms_target), C.byref(t)))
        return t.value
