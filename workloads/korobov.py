"""Choice of the Korobov generator `a` for a lattice size and dimension (R1).

The library embeds no lattice tables and none is typed from memory.  `a` is
found by a deterministic search that minimises the classical figure of merit

    P2(a) = -1 + (1/N) sum_{j<N} prod_{k<n} (1 + 2 pi^2 B2({j g_k / N})),
    B2(t) = t^2 - t + 1/6,   g_k = a^k mod N,

over the 64 odd candidates a_i = floor(N * frac(i*phi)) | 1, i = 1..64, phi the
golden ratio.  Results are cached in `korobov_table.json` beside this file,
written by `python -m workloads.korobov` (this script only; it calls neither the
oracle nor the CUDA path).  Parity needs only that both sides use the same `a`;
the figure of merit affects the integration error, not correctness.
"""
from __future__ import annotations

import json
import math
import os

import numpy as np

_TABLE_PATH = os.path.join(os.path.dirname(__file__), "korobov_table.json")
_PHI = (1.0 + math.sqrt(5.0)) / 2.0


def candidates(n_lattice: int):
    out = []
    for i in range(1, 65):
        a = int(n_lattice * ((i * _PHI) % 1.0)) | 1
        a %= n_lattice
        if a > 1 and a not in out:
            out.append(a)
    return out or [1]


def p2_merit(a: int, n_lattice: int, dim: int) -> float:
    j = np.arange(n_lattice, dtype=np.uint64)
    prod = np.ones(n_lattice)
    g = 1
    for _ in range(dim):
        t = ((j * np.uint64(g)) % np.uint64(n_lattice)).astype(np.float64) / n_lattice
        prod *= 1.0 + 2.0 * math.pi ** 2 * (t * t - t + 1.0 / 6.0)
        g = (g * a) % n_lattice
    return float(prod.mean() - 1.0)


def search(n_lattice: int, dim: int) -> int:
    best, best_a = None, 1
    for a in candidates(n_lattice):
        m = p2_merit(a, n_lattice, dim)
        if best is None or m < best:
            best, best_a = m, a
    return best_a


def _load():
    if os.path.exists(_TABLE_PATH):
        with open(_TABLE_PATH) as fh:
            return json.load(fh)
    return {}


def korobov_a(n_lattice: int, dim: int) -> int:
    """The cached generator for (N_L, n); searched on the spot if it is not in the table."""
    key = f"{n_lattice}:{dim}"
    tab = _load()
    if key in tab:
        return int(tab[key])
    return search(n_lattice, dim)


if __name__ == "__main__":
    table = _load()
    wanted = [(1 << 16, 4), (1 << 13, 4), (1 << 20, 6), (1 << 21, 8), (1 << 22, 7)]
    wanted += [(1 << m, d) for m in range(8, 19) for d in (1, 2, 3, 4, 6, 7, 8)]
    for n_lattice, dim in wanted:
        key = f"{n_lattice}:{dim}"
        if key not in table:
            table[key] = search(n_lattice, dim)
            print(key, table[key], flush=True)
            with open(_TABLE_PATH, "w") as fh:
                json.dump(table, fh, indent=0, sort_keys=True)
