"""Seeded synthetic objective tables (harness input; one array feeds oracle and GPU alike).

BASELINE.json: "objective fp32 = exp(sum of seeded N(0,0.3) per-value effects + seeded N(0,0.1)
pairwise terms)".  sigma is a standard deviation (reading A22).  The table is indexed by
valid rank, so it is built from a (parity-checked) valid-row table handed in by the caller.
"""
from __future__ import annotations
import numpy as np


def objective_table(rows: np.ndarray, m, seed: int = 0) -> np.ndarray:
    """rows: (V, >=n) uint8 index rows (padding columns ignored); m: values per parameter.

    obj[r] = float32(exp(sum_d E_d[idx_d] + sum_{d<e} Q_de[idx_d, idx_e])), accumulated in float64,
    main effects first (d ascending) then pairs in lexicographic (d, e) order.
    """
    n = len(m)
    rng = np.random.default_rng(np.random.SeedSequence([0xCA0, int(seed)]))
    E = [rng.normal(0.0, 0.3, size=int(m[d])) for d in range(n)]
    Q = {(d, e): rng.normal(0.0, 0.1, size=(int(m[d]), int(m[e])))
         for d in range(n) for e in range(d + 1, n)}
    idx = np.ascontiguousarray(rows[:, :n]).astype(np.intp)
    acc = np.zeros(idx.shape[0], dtype=np.float64)
    for d in range(n):
        acc += E[d][idx[:, d]]
    for d in range(n):
        for e in range(d + 1, n):
            acc += Q[(d, e)][idx[:, d], idx[:, e]]
    obj = np.exp(acc).astype(np.float32)
    assert np.all(np.isfinite(obj)) and np.all(obj > 0)
    return obj


def test_objective_37(V: int) -> np.ndarray:
    """obj[rank] = float(1 + (37*rank mod V)): the integer-valued table SURVEY.md's secondary pins use."""
    r = np.arange(V, dtype=np.int64)
    return (1 + (37 * r) % V).astype(np.float32)
