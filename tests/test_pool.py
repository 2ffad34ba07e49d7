"""CPU tests of the integration pool (paper_1511_03614_b200/pool.py): queue, partition, restartable store,
-part, totals; world size 2 over gloo.  The GPU is replaced by a stand-in context that returns numbers which
depend on the sector only; the GPU test of the pool is in test_gpu_parity.py."""
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_FAKE = r"""
import numpy as np
from dataclasses import dataclass, field
from paper_1511_03614_b200.binding import RESULT_DTYPE, Rule

@dataclass
class Sec:
    sector_id: int
    texts: list
    is_complex: bool = False
    deform_f_index: int = 0
    lam: float = 0.0

class FakeProg:
    def __init__(self, sectors): self.sectors, self.closed = sectors, False
    def close(self): self.closed = True

class FakeCtx:
    '''Stands in for binding.Context: the value of (sector, order) is a fixed function of the sector id.'''
    def __init__(self): self.compiled, self.integrated = [], []
    def compile(self, sectors, dim):
        self.compiled.append([s.sector_id for s in sectors]); return FakeProg(sectors)
    def integrate(self, prog, npoints, rule, seed, allow_nonfinite=False):
        assert not prog.closed
        out = np.zeros((len(prog.sectors), len(prog.sectors[0].texts)), dtype=RESULT_DTYPE)
        for i, s in enumerate(prog.sectors):
            for k in range(out.shape[1]):
                out[i, k] = (s.sector_id + 0.25 * k, 0.5 + s.sector_id, -k, 0.0, 0.0, npoints, 0)
        self.integrated.append([s.sector_id for s in prog.sectors]); return out

def sectors(n, K=2):
    return [Sec(100 + i, ["1;\n0;\nx[1]+%d.%d;\n|" % (i, k) for k in range(K)]) for i in range(n)]
"""


def _ns():
    ns = {}
    sys.path.insert(0, ROOT)
    exec(_FAKE, ns)
    return ns


def test_pool_queue_store_and_resume(tmp_path, lib):
    from paper_1511_03614_b200.pool import IntegrationPool, ResultStore
    ns = _ns()
    secs, rule = ns["sectors"](23), ns["Rule"](kind=1)
    costs = [(i * 7) % 5 + 1 for i in range(23)]
    path = str(tmp_path / "out.db")
    ctx = ns["FakeCtx"]()
    pool = IntegrationPool(ctx, secs, 1, rule, 1000, 7, store_path=path, group=5, costs=costs)
    assert not pool.run(max_groups=2)                       # a time limit: two groups of five, largest first
    assert pool.n_integrated == 10 and len(ctx.integrated) == 2
    assert all(costs[s - 100] >= 3 for g in ctx.integrated for s in g) and ctx.integrated[0] == [102, 107, 112, 117, 122]
    assert ctx.compiled == ctx.integrated                   # group 2 was handed to the compiler before group 1 ran; none beyond the limit
    with pytest.raises(RuntimeError):
        pool.totals()
    with open(path + ".rank0", "a") as fh:                  # the job was killed in the middle of a write
        fh.write('{"sig": "torn')
    # a new process continues from where it stopped: only the missing 13 are integrated
    ctx2 = ns["FakeCtx"]()
    pool2 = IntegrationPool(ctx2, secs, 1, rule, 1000, 7, store_path=path, group=5, costs=costs)
    assert pool2.run() and pool2.n_from_store == 10 and pool2.n_integrated == 13
    done_before = {s for g in ctx.integrated for s in g}
    assert not done_before & {s for g in ctx2.integrated for s in g}
    res = pool2.results()
    assert res.shape == (23, 2)
    for i in range(23):
        assert res[i, 1]["re"] == 100 + i + 0.25 and res[i, 0]["neval"] == 1000
    tot = pool2.totals()
    assert tot[0]["re"] == sum(100 + i for i in range(23))
    assert abs(tot[1]["re_err"] - np.sqrt(sum((0.5 + 100 + i) ** 2 for i in range(23)))) < 1e-9
    # other points / seed / texts: another signature, nothing is reused
    pool3 = IntegrationPool(ns["FakeCtx"](), secs, 1, rule, 2000, 7, store_path=path, group=50, costs=costs)
    assert len(pool3.pending()) == 23
    # a third run finds everything there and launches nothing
    ctx4 = ns["FakeCtx"]()
    pool4 = IntegrationPool(ctx4, secs, 1, rule, 1000, 7, store_path=path, group=5, costs=costs)
    assert pool4.run() and ctx4.integrated == [] and pool4.totals().tobytes() == tot.tobytes()


def test_pool_part_option(tmp_path, lib):
    """-part i/n: the parts are disjoint, cover everything, and their totals add up."""
    from paper_1511_03614_b200.pool import IntegrationPool
    ns = _ns()
    secs, rule = ns["sectors"](10), ns["Rule"](kind=1)
    seen, total = [], 0.0
    for i in (1, 2, 3):
        ctx = ns["FakeCtx"]()
        pool = IntegrationPool(ctx, secs, 1, rule, 500, 1, group=4, part=(i, 3))
        assert pool.run()
        seen += [s for g in ctx.integrated for s in g]
        total += pool.totals()[0]["re"]
    assert sorted(seen) == [100 + i for i in range(10)] and total == sum(100 + i for i in range(10))
    with pytest.raises(ValueError):
        IntegrationPool(ns["FakeCtx"](), secs, 1, rule, 500, 1, part=(4, 3))


_GLOO_POOL = r"""
import os, sys
import numpy as np
import torch.distributed as dist
sys.path.insert(0, {root!r})
exec(open({fake!r}).read())
from paper_1511_03614_b200.pool import IntegrationPool
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
secs, rule = sectors(17), Rule(kind=1)
costs = [(i * 5) % 7 + 1 for i in range(17)]
ctx = FakeCtx()
pool = IntegrationPool(ctx, secs, 1, rule, 1000, 3, store_path={store!r}, group=4, costs=costs, dist=dist)
assert pool.run()
mine = sorted(s for g in ctx.integrated for s in g)
res = pool.results()
assert res.shape == (17, 2) and all(res[i, 0]["re"] == 100 + i for i in range(17))
tot = pool.totals()
assert tot[0]["re"] == sum(100 + i for i in range(17))
load = sum(costs[s - 100] for s in mine)
print("ok", dist.get_rank(), len(mine), load)
dist.barrier()
dist.destroy_process_group()
"""


def test_pool_world_size_2_gloo(tmp_path):
    fake = tmp_path / "fake.py"
    fake.write_text(_FAKE)
    script = tmp_path / "w.py"
    port = 29500 + os.getpid() % 2000
    script.write_text(_GLOO_POOL.format(root=ROOT, fake=str(fake), port=port, store=str(tmp_path / "db")))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=180) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    n = [int(o.split()[2]) for o, _ in outs]
    loads = [int(o.split()[3]) for o, _ in outs]
    assert sum(n) == 17 and abs(loads[0] - loads[1]) <= 7       # every sector once, balanced by cost
    # both ranks wrote their own file; a single-process restart finds all 17 there
    sys.path.insert(0, ROOT)
    ns = {}
    exec(_FAKE, ns)
    from paper_1511_03614_b200.pool import IntegrationPool
    ctx = ns["FakeCtx"]()
    pool = IntegrationPool(ctx, ns["sectors"](17), 1, ns["Rule"](kind=1), 1000, 3, store_path=str(tmp_path / "db"), group=4,
                           costs=[(i * 5) % 7 + 1 for i in range(17)])
    assert pool.run() and ctx.integrated == []


# ------------------------------------------------------------------ bisection of the cube

def test_bisection_rewrites_the_text_correctly():
    """bisect_sector against the change of variables it stands for, through the ORACLE's parser and walker:
    part(t) = jacobian * f(x(t)), x_k = p t (lower) or 1 - (1-p) t (upper); the parts cover the cube once."""
    import numpy as np
    from oracle.evaluate import LD, evaluate, evaluate_with_magnitude
    from oracle.parser import parse
    from paper_1511_03614_b200.bisection import bisect_sector, bisect_text
    from workloads import SectorText, make_workload
    wl = make_workload("C2", nsectors=1, npoints=1 << 10)
    s = wl.sectors[0]
    parts = bisect_sector(s, [2, 5], points=[0.5, 0.25])    # dyadic: 1 - p is exact in the text as well
    assert [p.sector_id for p in parts] == [4 * s.sector_id + h for h in range(4)]
    assert parts[1].meta["halves"] == {2: "upper", 5: "lower"} and parts[2].meta["halves"] == {2: "lower", 5: "upper"}
    rng = np.random.default_rng(0)
    t = rng.random((50, wl.dim)).astype(LD)
    for h, part in enumerate(parts):
        x = t.copy()
        jac = LD(1)
        for bit, (k, p) in enumerate(((2, LD(0.5)), (5, LD(0.25)))):
            if (h >> bit) & 1:
                x[:, k - 1] = 1 - (1 - p) * t[:, k - 1]
                jac = jac * (1 - p)
            else:
                x[:, k - 1] = p * t[:, k - 1]
                jac = jac * p
        for text, ptext in zip(s.texts, part.texts):
            ref, mag = evaluate_with_magnitude(parse(text), x)
            got = evaluate(parse(ptext), t)
            assert np.all(np.abs(got - jac * ref) <= 1e-17 * jac * mag)
    # a 1-D integrand integrated exactly: x^3 over [0,1] = 1/4 from the two parts' antiderivatives
    lo, up = (parse(bisect_text("1;\n0;\np[x[1],3];\n|", {1: (0.25, u)})) for u in (False, True))
    nodes, weights = np.polynomial.legendre.leggauss(4)
    tt = ((nodes + 1) / 2)[:, None].astype(LD)
    total = sum(float(np.sum(weights / 2 * evaluate(prog, tt).astype(float))) for prog in (lo, up))
    assert abs(total - 0.25) < 1e-15
    # errors
    import pytest
    with pytest.raises(ValueError):
        bisect_sector(s, [2, 2])
    with pytest.raises(ValueError):
        bisect_sector(s, [wl.dim + 1])
    with pytest.raises(ValueError):
        bisect_sector(s, [1], points=1.0)
    tiny = bisect_sector(SectorText(sector_id=0, texts=["1;\n0;\nx[1];\n|"]), [1], points=1e-7)   # exponent literals parse
    assert abs(float(evaluate(parse(tiny[0].texts[0]), np.array([[0.5]], dtype=LD))[0]) - 0.5e-14) < 1e-28


class _StubDist:
    """torch.distributed's query functions for a rank that never talks to anybody (the frozen-worker tests)."""

    def __init__(self, rank, world):
        self.rank, self.world = rank, world

    def is_initialized(self):
        return True

    def get_rank(self):
        return self.rank

    def get_world_size(self):
        return self.world


def test_pool_resubmits_the_work_of_frozen_ranks(tmp_path, lib):
    """a rank that froze mid-way and one that never came up; the surviving rank takes their sectors
    over through the store files, and the totals are those of an undisturbed job."""
    import time
    from paper_1511_03614_b200.pool import IntegrationPool
    ns = _ns()
    secs, rule = ns["sectors"](20), ns["Rule"](kind=1)
    costs = [(i * 3) % 7 + 1 for i in range(20)]
    path = str(tmp_path / "db")
    mk = lambda r, ctx: IntegrationPool(ctx, secs, 1, rule, 1000, 9, store_path=path, group=2, costs=costs, dist=_StubDist(r, 3))
    ctx1 = ns["FakeCtx"]()
    p1 = mk(1, ctx1)
    assert not p1.run(max_groups=1)                       # rank 1 stores one group, then hangs; rank 2 never starts
    ctx0 = ns["FakeCtx"]()
    p0 = mk(0, ctx0)
    assert p0.run() and p0.frozen_ranks(stale_after=3600.0) == []      # nobody is late yet
    with pytest.raises(RuntimeError):
        p0.results(collective=False)
    time.sleep(0.05)
    assert p0.frozen_ranks(stale_after=0.01) == [1, 2]
    done1 = {s for g in ctx1.integrated for s in g}
    n = p0.adopt([1, 2])
    owed = set(100 + j for r in (1, 2) for j in p0.shares[r]) - done1
    adopted = [s for g in ctx0.integrated for s in g][len(p0.my_local):]
    assert n == len(owed) == p0.n_adopted and set(adopted) == owed
    assert [costs[s - 100] for s in adopted] == sorted(costs[s - 100] for s in adopted)    # cheapest first
    res = p0.results(collective=False)
    assert all(res[i, 0]["re"] == 100 + i for i in range(20))
    assert p0.totals(collective=False)[0]["re"] == sum(100 + i for i in range(20))
    assert p0.frozen_ranks(stale_after=0.0) == []         # nothing is owed any more
    # the slow rank wakes up: everything it owed is in the store, it computes nothing and sees the same totals
    ctx1b = ns["FakeCtx"]()
    p1b = mk(1, ctx1b)
    assert p1b.run() and ctx1b.integrated == []
    assert p1b.totals(collective=False).tobytes() == p0.totals(collective=False).tobytes()
    # run_to_completion: own share, then the frozen ranks' (a fresh store)
    path2 = str(tmp_path / "db2")
    ctx = ns["FakeCtx"]()
    p = IntegrationPool(ctx, secs, 1, rule, 1000, 9, store_path=path2, group=4, costs=costs, dist=_StubDist(2, 3))
    assert p.run_to_completion(stale_after=0.0, poll=0.01, timeout=5.0)
    assert sorted(s for g in ctx.integrated for s in g) == [100 + i for i in range(20)] and p.n_adopted == 20 - len(p.my_local)


# ------------------------------------------------------------------ few, huge sectors: shifts split over ranks

_GLOO_SHIFTS = r"""
import sys
import numpy as np
import torch.distributed as dist
sys.path.insert(0, {root!r})
from paper_1511_03614_b200.sharding import integrate_split_shifts, split_shifts
from paper_1511_03614_b200.binding import Rule
world = {world}
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=world)

class Prog:
    nsectors = 3

class Ctx:
    '''stands in for binding.Context: the sums of (sector, shift) are a fixed function of both'''
    def __init__(self): self.asked = []
    def partial_sums_shifts(self, prog, npoints, rule, seed, first, count, sectors=None, tier=-1):
        self.asked.append((first, count))
        out = np.zeros((3, count, 2, 1, 2))
        for s in range(3):
            for r in range(count):
                out[s, r] = 1000 * s + 10 * (first + r) + np.arange(4).reshape(2, 1, 2)
        return out, np.array([first, 0, count], dtype=np.uint64)
    def estimate_from_sums(self, prog, sums, n_per_shift, nonfinite=None, sectors=None, allow_nonfinite=False):
        return sums, nonfinite, n_per_shift

R = {R}
ctx = Ctx()
sums, nf, nps = integrate_split_shifts(ctx, Prog(), 8 * R, Rule(kind=0, n_shifts=R), 1, dist=dist)
shares = split_shifts(R, world)
assert ctx.asked == ([shares[dist.get_rank()]] if shares[dist.get_rank()][1] else [])
assert sums.shape == (3, R, 2, 1, 2) and nps == 8
for s in range(3):
    for r in range(R):
        assert np.array_equal(sums[s, r], 1000 * s + 10 * r + np.arange(4).reshape(2, 1, 2))
assert nf.tolist() == [sum(f for f, c in shares if c), 0, R]
print("ok")
dist.barrier()
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,R", [(2, 8), (3, 2)])
def test_shifts_split_over_ranks_gloo(tmp_path, world, R):
    """sharding.integrate_split_shifts: every rank asks for its share of the shifts only, the gathered rows are in
    shift order on every rank, non-finite counts add up; also with more ranks than shifts."""
    from paper_1511_03614_b200.sharding import split_shifts
    assert split_shifts(8, 3) == [(0, 3), (3, 3), (6, 2)] and split_shifts(2, 3) == [(0, 1), (1, 1), (2, 0)]
    script = tmp_path / "s.py"
    port = 31500 + (os.getpid() + 7 * world) % 2000
    script.write_text(_GLOO_SHIFTS.format(root=ROOT, port=port, world=world, R=R))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(world)]
    outs = [p.communicate(timeout=180) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0 and "ok" in o, e[-2000:]
