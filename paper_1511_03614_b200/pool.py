"""Integration pool: the queue over the integrands of a job, with restartable results.

The paper's CIntegratePool "reads the integrands from the integration database ... creating an
integration queue, while the integration binaries work on particular expressions";
on a cluster a master "distributes the jobs to the slave nodes"; with `-continue` all
intermediate results are saved in the output database, so that after a crash or a timeout "the code
can afterwards continue from the moment it stopped at"; `-part i/n` works
on the i-th of n parts of the integrands; per order the results are summed with the
errors in mean square.

Here the integrands are the sectors of a job, the worker is one process per GPU (`torch.distributed`
rank) calling the C ABI, and this module is the host-side queue around it -- no arithmetic of the
method, only which sectors go where and when:

  * partition: the part's sectors are dealt to the ranks by longest processing time on a cost per
    sector (sharding.partition_sectors); every rank computes the same plan, nothing is sent;
  * queue: a rank works its share off in groups of `group` sectors, largest first.  Group g+1 is
    handed to fiesta_compile BEFORE group g is integrated, so the background assembly of its
    native kernels overlaps the integration of the group in front of it;
  * store: after every group the per-(sector, order) records are appended to a JSON-lines file and
    flushed to disk; a record carries the signature of what produced it (rule, points, seed, the
    sector's texts), so a later run skips exactly the work that is already there;
  * totals: when every sector of the part is there, the ranks exchange their records once
    (sharding.gather_results) and fiesta_combine sums per order;
  * frozen workers: "if some of the slave jobs become frozen during the integration, FIESTA is
    capable of resubmitting their tasks to other nodes"; jobs whose integrators "are initialized
    improperly" are passed over.  Here every rank can read every rank's store file
    (a shared file system): a rank that still owes sectors and whose file has not grown for
    `stale_after` seconds -- or was never created -- counts as frozen (frozen_ranks), and a rank
    that is through with its own share takes those sectors over (adopt), cheapest first, i.e. from
    the far end of the owner's queue.  A sector's result does not depend on who computes it (same
    sector id, seed and rule: the same bits), so a slow owner that finishes after all merely writes
    a duplicate record.  With a dead rank a collective would hang: results(collective=False) reads
    the part's records from the store files instead.
"""
from __future__ import annotations

import ctypes as C
import hashlib
import json
import os
import time

import numpy as np

from .binding import RESULT_DTYPE, FiestaError, E_NONFINITE, load_library
from .sharding import gather_results, partition_sectors


def _signature(sector, dim, rule, npoints, seed):
    h = hashlib.sha256()
    h.update(repr((dim, rule.kind, rule.n_shifts, rule.korobov_a, tuple(rule.genvec or ()), rule.periodize_r,
                   rule.vegas_bins, rule.vegas_iters, rule.vegas_alpha, int(npoints), int(seed),
                   int(sector.sector_id), bool(sector.is_complex), int(sector.deform_f_index), float(sector.lam))).encode())
    for t in sector.texts:
        h.update(t.encode())
    return h.hexdigest()[:24]


class ResultStore:
    """Append-only JSON-lines store of per-(sector, order) results (PAPER.md:146 `-continue`, :489 `-save_all`)."""

    FIELDS = ("re", "re_err", "im", "im_err", "chi2", "neval", "n_nonfinite")

    def __init__(self, path, rank=0):
        self.path = path
        self.mine = None if path is None else f"{path}.rank{rank}"
        self.rows = {}          # signature -> {order: record dict}
        if path is not None:
            d = os.path.dirname(os.path.abspath(path))
            os.makedirs(d, exist_ok=True)
            base = os.path.basename(path)
            for name in sorted(os.listdir(d)):      # every rank's file: a restart may use another number of ranks
                if name.startswith(base + ".rank"):
                    self._load(os.path.join(d, name))

    def refresh(self):
        """Read every rank's file again: what the other ranks have stored since this object was made."""
        if self.path is None:
            return
        d = os.path.dirname(os.path.abspath(self.path))
        base = os.path.basename(self.path)
        for name in sorted(os.listdir(d)):
            if name.startswith(base + ".rank"):
                self._load(os.path.join(d, name))

    def age(self, rank, now=None):
        """Seconds since rank's file was last written; None if it does not exist."""
        f = f"{self.path}.rank{rank}"
        if self.path is None or not os.path.exists(f):
            return None
        return (time.time() if now is None else now) - os.path.getmtime(f)

    def _load(self, file):
        with open(file) as fh:
            for line in fh:
                try:
                    rec = json.loads(line)
                    self.rows.setdefault(rec["sig"], {})[int(rec["k"])] = rec
                except (ValueError, KeyError):
                    continue                          # a torn last line of an interrupted run

    def get(self, sig, K):
        """The stored [K] records of a sector, or None if any order is missing."""
        have = self.rows.get(sig, {})
        if any(k not in have for k in range(K)):
            return None
        out = np.zeros(K, dtype=RESULT_DTYPE)
        for k in range(K):
            for f in self.FIELDS:
                out[k][f] = have[k][f]
        return out

    def put_group(self, sigs, sector_ids, results):
        """results [nsec][K]: append and flush to disk before returning."""
        lines = []
        for sig, sid, row in zip(sigs, sector_ids, results):
            for k in range(row.shape[0]):
                rec = {"sig": sig, "sector_id": int(sid), "k": k}
                for f in self.FIELDS:
                    v = row[k][f]
                    rec[f] = int(v) if f in ("neval", "n_nonfinite") else float(v)
                self.rows.setdefault(sig, {})[k] = rec
                lines.append(json.dumps(rec))
        if self.mine is not None and lines:
            torn = False                                  # a killed run may have left half a line: start a new one
            if os.path.exists(self.mine) and os.path.getsize(self.mine) > 0:
                with open(self.mine, "rb") as fh:
                    fh.seek(-1, os.SEEK_END)
                    torn = fh.read(1) != b"\n"
            with open(self.mine, "a") as fh:
                fh.write(("\n" if torn else "") + "\n".join(lines) + "\n")
                fh.flush()
                os.fsync(fh.fileno())


def combine(per_sector):
    """fiesta_combine: sum over sectors, errors in mean square.  Host arithmetic of the library."""
    per_sector = np.ascontiguousarray(per_sector, dtype=RESULT_DTYPE)
    S, K = per_sector.shape
    tot = np.zeros(K, dtype=RESULT_DTYPE)
    rc = load_library().fiesta_combine(per_sector.ctypes.data_as(C.c_void_p), S, K, tot.ctypes.data_as(C.c_void_p))
    if rc:
        raise FiestaError(rc, "fiesta_combine")
    return tot


class IntegrationPool:
    """Queue over the sectors of a job on this rank's GPU; see the module docstring.

    ctx: binding.Context (anything with compile(sectors, dim) and integrate(prog, npoints, rule, seed, ...)).
    sectors: objects with .sector_id, .texts, .is_complex, .deform_f_index, .lam (workloads.SectorText).
    costs: per-sector work estimate for the partition (default: text length x points).
    part: (i, n), 1-based: only the i-th of n contiguous parts of the sectors (PAPER.md:487 `-part`).
    dist: torch.distributed (initialised) or None; device: where the gather's tensors live."""

    def __init__(self, ctx, sectors, dim, rule, npoints, seed, store_path=None, group=64, part=None, costs=None,
                 dist=None, device="cpu"):
        self.ctx, self.dim, self.rule, self.npoints, self.seed = ctx, dim, rule, int(npoints), int(seed)
        self.dist = dist if (dist is not None and dist.is_initialized() and dist.get_world_size() > 1) else None
        self.rank = self.dist.get_rank() if self.dist else 0
        self.world = self.dist.get_world_size() if self.dist else 1
        self.device = device
        self.group = max(1, int(group))
        n = len(sectors)
        lo, hi = 0, n
        if part is not None:
            i, parts = part
            if not (1 <= i <= parts):
                raise ValueError("part must be (i, n) with 1 <= i <= n")
            lo, hi = (i - 1) * n // parts, i * n // parts
        self.indices = list(range(lo, hi))                 # positions in `sectors` this job covers
        self.sectors = sectors
        K = {len(sectors[i].texts) for i in self.indices}
        if len(K) > 1:
            raise ValueError("all sectors of a pool job must have the same number of orders")
        self.K = K.pop() if K else 0
        if costs is None:
            costs = [sum(len(t) for t in s.texts) * float(npoints) for s in sectors]
        self.costs = [float(costs[i]) for i in self.indices]
        shares = partition_sectors(self.costs, self.world)
        self.shares = [sorted(sh, key=lambda j: (-self.costs[j], j)) for sh in shares]  # every rank's queue, largest first
        self.my_local = self.shares[self.rank]
        self.started = time.time()
        self.n_adopted = 0                                  # sectors taken over from frozen ranks
        self.sigs = {j: _signature(sectors[self.indices[j]], dim, rule, npoints, seed) for j in range(len(self.indices))}
        self.store = ResultStore(store_path, self.rank)
        self.n_integrated = 0                               # sectors this object sent to the GPU
        self.n_from_store = 0

    def pending(self):
        """This rank's sectors (local numbers) that are not in the store yet, in queue order."""
        return [j for j in self.my_local if self.store.get(self.sigs[j], self.K) is None]

    def run(self, max_groups=None):
        """Work the queue off (at most max_groups groups: a time limit).  Returns True when this rank is done."""
        todo = self.pending()
        self.n_from_store = len(self.my_local) - len(todo)
        self._work(todo, max_groups)
        return not self.pending()

    def frozen_ranks(self, stale_after):
        """Other ranks that still owe sectors and whose store file has not been written for `stale_after`
        seconds -- or does not exist `stale_after` seconds after this pool was made (a worker that never
        came up).  Reads the store files again first."""
        if self.store.path is None:
            raise RuntimeError("frozen workers are recognised by their store files: the pool needs a store_path")
        self.store.refresh()
        now = time.time()
        out = []
        for r in range(self.world):
            if r == self.rank or all(self.store.get(self.sigs[j], self.K) is not None for j in self.shares[r]):
                continue
            age = self.store.age(r, now)
            if (now - self.started if age is None else age) >= stale_after:
                out.append(r)
        return out

    def adopt(self, ranks, max_groups=None):
        """Integrate what the given (frozen) ranks still owe, cheapest sectors first -- the far end of their
        queues, which a merely slow owner reaches last.  Returns the number of sectors taken over."""
        self.store.refresh()
        todo = [j for r in ranks for j in self.shares[r] if self.store.get(self.sigs[j], self.K) is None]
        todo.sort(key=lambda j: (self.costs[j], j))
        before = self.n_integrated
        self._work(todo, max_groups)
        self.n_adopted += self.n_integrated - before
        return self.n_integrated - before

    def run_to_completion(self, stale_after, poll=1.0, timeout=None):
        """run(), then watch the other ranks: adopt the sectors of those that freeze, until the whole part is in
        the store (True) or `timeout` seconds have passed (False)."""
        self.run()
        t0 = time.time()
        while True:
            self.store.refresh()
            if all(self.store.get(self.sigs[j], self.K) is not None for j in range(len(self.indices))):
                return True
            frozen = self.frozen_ranks(stale_after)
            if frozen:
                self.adopt(frozen)
                continue
            if timeout is not None and time.time() - t0 > timeout:
                return False
            time.sleep(poll)

    def _work(self, todo, max_groups=None):
        groups = [todo[i:i + self.group] for i in range(0, len(todo), self.group)]
        if max_groups is not None:
            groups = groups[:max_groups]
        progs = {}

        def compiled(g):
            if g not in progs and g < len(groups):
                progs[g] = self.ctx.compile([self.sectors[self.indices[j]] for j in groups[g]], self.dim)
            return progs.get(g)

        for g, members in enumerate(groups):
            prog = compiled(g)
            compiled(g + 1)                                # its kernels are assembled while group g integrates
            res = self.ctx.integrate(prog, self.npoints, self.rule, self.seed, allow_nonfinite=True)
            self.store.put_group([self.sigs[j] for j in members], [self.sectors[self.indices[j]].sector_id for j in members], res)
            self.n_integrated += len(members)
            close = getattr(progs.pop(g), "close", None)
            if close:
                close()

    def results(self, collective=True):
        """[sectors of the part][K] of ALL ranks; raises if some sector is not there yet.  collective=True: one
        gather of every rank's own share; False: from the store files alone (no rank waits for another)."""
        if not collective:
            self.store.refresh()
            out = np.zeros((len(self.indices), self.K), dtype=RESULT_DTYPE)
            for j in range(len(self.indices)):
                row = self.store.get(self.sigs[j], self.K)
                if row is None:
                    raise RuntimeError(f"sector {self.sectors[self.indices[j]].sector_id} has not been integrated yet")
                out[j] = row
            return out
        mine = self.my_local
        local = np.zeros((len(mine), self.K), dtype=RESULT_DTYPE)
        for a, j in enumerate(mine):
            row = self.store.get(self.sigs[j], self.K)
            if row is None:
                raise RuntimeError(f"sector {self.sectors[self.indices[j]].sector_id} has not been integrated yet")
            local[a] = row
        return gather_results(local, mine, len(self.indices), self.dist, self.device)

    def totals(self, collective=True):
        """Per order: sum over the part's sectors, errors in mean square."""
        return combine(self.results(collective))
