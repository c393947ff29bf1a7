"""Seeded generators for BASELINE.json's five DF-JK configs (recipe: DESIGN.md "Input recipe").

Only random draws, a QR for orthonormal columns, and the decay envelope of B live here; nothing
of Eq. 12-17.  All arrays are C-contiguous float64 numpy arrays on the host.

Recipe
  B_packed[P, idx(mu,nu)] = z * exp(-|mu-nu| / L) / sqrt(naux),  z ~ N(0,1),
      z = default_rng(seedB).standard_normal((naux, npair)) drawn row-major (row chunks give the
      identical stream), idx(mu,nu) = mu(mu+1)/2 + nu for mu >= nu (numpy.tril_indices order).
  C: Q from numpy.linalg.qr(default_rng(seedC).standard_normal((nao, nao))), leading columns.
  Seeds: config k = 1..5 -> seedB = 1000+k, seedC = 2000+k, seedC2 = 3000+k, seedO = 4000+k.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np


def npair_of(nao: int) -> int:
    return nao * (nao + 1) // 2


# name -> (k, nao, naux, nocc per set, decay length L)
CONFIGS = {
    "tiny": dict(k=1, nao=48, naux=160, nocc=[12], L=8.0),
    "small": dict(k=2, nao=300, naux=1000, nocc=[80], L=20.0),
    "medium": dict(k=3, nao=600, naux=2000, nocc=[150, 140], L=40.0),
    "large": dict(k=4, nao=1200, naux=4000, nocc=[300], L=80.0),
    "lasscf": dict(k=5, nao=1200, naux=4000, nocc=[290, 8, 8, 8, 8, 8], L=80.0),
}


@dataclass
class DFJKInputs:
    name: str
    nao: int
    naux: int
    nocc: List[int]                 # per set
    B_packed: Optional[np.ndarray]  # (naux, npair) or None when make_config(..., with_B=False)
    C: List[np.ndarray]             # per set, (nao, nocc[s]) row-major
    occ: List[np.ndarray]           # per set, (nocc[s],)
    L: float = 0.0
    seeds: dict = field(default_factory=dict)

    @property
    def nset(self) -> int:
        return len(self.nocc)

    @property
    def npair(self) -> int:
        return npair_of(self.nao)

    def C_concat(self) -> np.ndarray:
        """Blocks [C_0 | C_1 | ...] laid out one after another (each block row-major nao x nocc[s])."""
        return np.concatenate([np.ascontiguousarray(c).ravel() for c in self.C]) if self.C else np.zeros(0)

    def occ_concat(self) -> np.ndarray:
        return np.concatenate(self.occ) if self.occ else np.zeros(0)


def decay_envelope(nao: int, naux: int, L: float) -> np.ndarray:
    """exp(-|mu-nu|/L)/sqrt(naux) for every packed pair, in tril_indices order."""
    mu, nu = np.tril_indices(nao)
    return np.exp(-np.abs(mu - nu) / L) / np.sqrt(naux)


def make_B_packed(nao: int, naux: int, L: float, seedB: int, rows: Optional[int] = None,
                  chunk_rows: int = 64, out: Optional[np.ndarray] = None) -> np.ndarray:
    """Packed B, first ``rows`` aux rows (default all).  Row-chunked draws equal one big draw."""
    npair = npair_of(nao)
    rows = naux if rows is None else rows
    env = decay_envelope(nao, naux, L)
    rng = np.random.default_rng(seedB)
    B = np.empty((rows, npair), dtype=np.float64) if out is None else out
    assert B.shape == (rows, npair) and B.dtype == np.float64 and B.flags.c_contiguous
    for r0 in range(0, rows, chunk_rows):
        r1 = min(rows, r0 + chunk_rows)
        rng.standard_normal(out=B[r0:r1])
        B[r0:r1] *= env
    return B


def _q_of(nao: int, seed: int) -> np.ndarray:
    q, _ = np.linalg.qr(np.random.default_rng(seed).standard_normal((nao, nao)))
    return q


def make_orbitals(name: str, all_columns: bool = False):
    """(C list, occ list) of a named config; with all_columns the whole orthonormal nao x nao
    matrix Q the columns are taken from (seedC), e.g. as MO coefficients for AO2MO."""
    cfg = CONFIGS[name]
    k, nao, nocc = cfg["k"], cfg["nao"], cfg["nocc"]
    seedC, seedC2, seedO = 2000 + k, 3000 + k, 4000 + k
    if all_columns:
        return _q_of(nao, seedC)
    if name == "medium":
        qa, qb = _q_of(nao, seedC), _q_of(nao, seedC2)
        C = [np.ascontiguousarray(qa[:, :nocc[0]]), np.ascontiguousarray(qb[:, :nocc[1]])]
        occ = [np.ones(nocc[0]), np.ones(nocc[1])]
    elif name == "lasscf":
        q = _q_of(nao, seedC)
        act = np.random.default_rng(seedO).uniform(0.0, 2.0, 40)
        act *= 22.0 / act.sum()
        C, occ, c0 = [], [], 0
        for s, n in enumerate(nocc):
            C.append(np.ascontiguousarray(q[:, c0:c0 + n]))
            occ.append(np.full(n, 2.0) if s == 0 else act[(s - 1) * 8:s * 8].copy())
            c0 += n
    else:
        q = _q_of(nao, seedC)
        C = [np.ascontiguousarray(q[:, :nocc[0]])]
        occ = [np.full(nocc[0], 2.0)]
    return C, occ


def make_config(name: str, with_B: bool = True, aux_rows: Optional[int] = None) -> DFJKInputs:
    """Inputs of a named config.  ``aux_rows`` keeps only the first rows of B (same stream);
    the 1/sqrt(naux) scale stays that of the full config so samples are slices of the real B."""
    cfg = CONFIGS[name]
    k, nao, naux, L = cfg["k"], cfg["nao"], cfg["naux"], cfg["L"]
    C, occ = make_orbitals(name)
    B = make_B_packed(nao, naux, L, 1000 + k, rows=aux_rows) if with_B else None
    return DFJKInputs(name=name, nao=nao, naux=naux if aux_rows is None else aux_rows,
                      nocc=list(cfg["nocc"]), B_packed=B, C=C, occ=occ, L=L,
                      seeds=dict(seedB=1000 + k, seedC=2000 + k, seedC2=3000 + k, seedO=4000 + k))


def make_random(nao: int, naux: int, nocc: List[int], seed: int, L: float = 0.0,
                orthonormal: bool = False) -> DFJKInputs:
    """Free-form seeded inputs for edge-case tests: Gaussian B (optionally with the decay
    envelope), Gaussian non-orthonormal C unless asked otherwise, occupations uniform in [0,2]."""
    rng = np.random.default_rng(seed)
    npair = npair_of(nao)
    B = rng.standard_normal((naux, npair))
    if L > 0:
        B *= decay_envelope(nao, max(naux, 1), L)
    C, occ = [], []
    for n in nocc:
        c = rng.standard_normal((nao, n))
        if orthonormal and n > 0:
            c, _ = np.linalg.qr(c)
        C.append(np.ascontiguousarray(c))
        occ.append(rng.uniform(0.0, 2.0, n))
    return DFJKInputs(name=f"random{seed}", nao=nao, naux=naux, nocc=list(nocc), B_packed=B, C=C,
                      occ=occ, L=L, seeds=dict(seed=seed))
