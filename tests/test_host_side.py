"""CPU-only tests of the host side: the C-ABI library loads and exports every declared symbol,
the host-arithmetic entry point fiesta_combine, no-GPU failure is loud, and the multi-GPU
sharding logic (world_size 2 over gloo).  No compute calls on a device here."""
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "fiesta_b200.h")).read()
    declared = set(re.findall(r"\b(fiesta_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 19
    handle = lib.load_library()
    for name in declared:
        assert getattr(handle, name) is not None, name
    assert declared == set(lib.exported_symbols())
    out = subprocess.run(["nm", "-D", "--defined-only", lib.LIB_PATH], capture_output=True, text=True).stdout
    exported = set(re.findall(r" T (fiesta_[a-z0-9_]+)", out))
    assert declared <= exported


def test_library_is_built_for_sm100a(lib):
    out = subprocess.run(["cuobjdump", "-lelf", lib.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out


def test_struct_layouts_match_header(lib):
    assert lib.RESULT_DTYPE.itemsize == 56      # 5 doubles + 2 uint64
    assert lib.INFO_DTYPE.itemsize == 48        # 9 int32 (+pad) + 1 double


def test_combine_mean_square(lib):
    """values add, errors add in mean square."""
    rng = np.random.default_rng(0)
    S, K = 7, 3
    per = np.zeros((S, K), dtype=lib.RESULT_DTYPE)
    for f in ("re", "re_err", "im", "im_err", "chi2"):
        per[f] = rng.random((S, K))
    per["neval"] = 100
    per["n_nonfinite"] = rng.integers(0, 3, (S, K))
    tot = np.zeros(K, dtype=lib.RESULT_DTYPE)
    from paper_1511_03614_b200.binding import _ptr
    rc = lib.load_library().fiesta_combine(_ptr(per), S, K, _ptr(tot))
    assert rc == 0
    assert np.allclose(tot["re"], per["re"].sum(axis=0), rtol=1e-15)
    assert np.allclose(tot["im"], per["im"].sum(axis=0), rtol=1e-15)
    assert np.allclose(tot["re_err"], np.sqrt((per["re_err"] ** 2).sum(axis=0)), rtol=1e-15)
    assert np.allclose(tot["im_err"], np.sqrt((per["im_err"] ** 2).sum(axis=0)), rtol=1e-15)
    assert np.all(tot["neval"] == 100 * S) and np.all(tot["n_nonfinite"] == per["n_nonfinite"].sum(axis=0))
    assert lib.load_library().fiesta_combine(None, S, K, _ptr(tot)) == -7


def test_no_gpu_fails_loudly(lib):
    """No CPU fallback: without an sm_100 device the context cannot be created."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(lib.FiestaError) as ei:
        lib.Context(0)
    assert ei.value.code == -5


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1511_03614_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cpp", ".cu", ".cuh", ".h", ".hpp", ".inc")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
                assert "oracle/" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_1511_03614_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "`paper_1511_03614_b200/`", ""), f


# ------------------------------------------------------------------------------ sharding

def test_partition_is_balanced_and_complete():
    from paper_1511_03614_b200.sharding import partition_sectors
    rng = np.random.default_rng(1)
    costs = rng.integers(500, 1500, 2000).astype(float)
    for world in (1, 2, 3, 8):
        parts = partition_sectors(costs, world)
        allidx = sorted(i for p in parts for i in p)
        assert allidx == list(range(2000))
        loads = [costs[p].sum() for p in parts]
        assert max(loads) - min(loads) <= costs.max()
    assert partition_sectors([5.0], 4) == [[0], [], [], []]
    assert partition_sectors([], 2) == [[], []]


_GLOO_WORKER = r"""
import os, sys
import numpy as np
import torch.distributed as dist
sys.path.insert(0, {root!r})
from paper_1511_03614_b200.sharding import partition_sectors, gather_results, max_over_ranks
from paper_1511_03614_b200.binding import RESULT_DTYPE
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
S, K = 11, 3
costs = [(i * 7) % 5 + 1 for i in range(S)]
mine = partition_sectors(costs, 2)[rank]
local = np.zeros((len(mine), K), dtype=RESULT_DTYPE)
for a, s in enumerate(mine):          # a stand-in for this rank's fiesta_integrate output
    for k in range(K):
        local[a, k] = (s + 0.1 * k, 0.01 * s, -s, 0.5, k, 1000 + s, s % 2)
full = gather_results(local, mine, S, dist)
for s in range(S):
    for k in range(K):
        assert full[s, k]["re"] == s + 0.1 * k and full[s, k]["neval"] == 1000 + s and full[s, k]["im"] == -s
t = max_over_ranks(1.0 + rank, dist)
assert t == 2.0
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_gather_results_world_size_2_gloo(tmp_path):
    port = 29500 + (os.getpid() % 2000)
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {r}" in o, o


# ------------------------------------------------------------------------------ native tier (host part)

def _count(ptx, op):
    return sum(1 for ln in ptx.splitlines() if ln.strip().startswith(op + " "))


def test_native_lowering_of_the_paper_example(lib):
    """PAPER.md:517-519, `1; 0; x[1]+0.2;`: the whole program is one add per point of the batch, then
    the accumulation of the single output; the module assembles for sm_100a without a GPU."""
    from workloads import SectorText
    ptx, nbytes = lib.native_assemble(SectorText(sector_id=0, texts=["1;\n0;\nx[1]+0.2;\n|"]), 1)
    assert nbytes > 10000
    body = [ln.strip() for ln in ptx.splitlines()]
    adds = [ln for ln in body if ln.startswith(("add.rn.f64 %fxa", "fma.rn.f64 %fxa"))]
    assert len(adds) == 2 and all("%x0_" in ln for ln in adds)            # 2 points per pass, x[1] = register file X[0]
    assert body[0].startswith(".const .align 8 .f64 fxj_const[1] = {0d3FC999999999999A}")   # 0.2, bit pattern
    movs = [ln for ln in body if ln.startswith("mov.f64 %fxa") and ln.endswith("%fxc;")]
    assert len(movs) == 2 and "ld.const.f64 %fxc, [fxj_const+0];" in body
    assert _count(ptx, "st.shared.f64") == 2 and _count(ptx, "setp.eq.u32 %fxf,") == 2   # sum g, sum g^2; non-finite count


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C5"])
def test_native_lowering_keeps_every_operation(lib, name):
    """The generated body has exactly the program's arithmetic (x 2 points per pass): every FMA explicit, every
    other operation with its rounding; logs and exps become calls; K outputs are accumulated."""
    from workloads import make_workload
    wl = make_workload(name, nsectors=2, npoints=1 << 10)
    for s in wl.sectors:
        ptx, nbytes = lib.native_assemble(s, wl.dim)
        assert nbytes > 10000
        assert "fma.f64" not in ptx and "mul.f64" not in ptx and "add.f64" not in ptx     # nothing left to contract
        K = len(s.texts)
        n_out = _count(ptx, "setp.eq.u32 %fxf,")
        assert n_out == 2 * K
        n_fma = _count(ptx, "fma.rn.f64") - n_out          # minus sum g^2 of the sink
        n_mul = _count(ptx, "mul.rn.f64") - n_out          # minus g = W*o
        n_add = _count(ptx, "add.rn.f64") + _count(ptx, "sub.rn.f64") - n_out
        n_div = _count(ptx, "div.rn.f64")
        n_call = ptx.count("call.uni")
        assert min(n_fma, n_mul, n_add) >= 0 and (n_fma + n_mul + n_add + n_div + n_call) % 2 == 0
        assert n_fma > 0 and n_call % 2 == 0


def test_native_assemble_rejects_complex_and_bad_text(lib):
    from workloads import SectorText
    with pytest.raises(lib.FiestaError):
        lib.native_assemble(SectorText(sector_id=0, texts=["1;\n0;\nx[1];\n|"], is_complex=True), 1)
    with pytest.raises(lib.FiestaError) as e:
        lib.native_assemble(SectorText(sector_id=0, texts=["1;\n0;\nx[1]+;\n|"]), 1)
    assert "line" in str(e.value) or "expected" in str(e.value) or len(str(e.value)) > 0
