"""ctypes/numpy marshalling for oracle/dfjk_oracle.c.  No arithmetic of the method lives here."""
from __future__ import annotations

import ctypes as ct
import os
from typing import List, Optional, Sequence, Tuple

import numpy as np

from . import build as _build

_lib = None
_dp = ct.POINTER(ct.c_double)
_ip = ct.POINTER(ct.c_int)


def _load():
    global _lib
    if _lib is None:
        # many short parallel regions: sleeping waiters beat spinning ones on shared hosts
        os.environ.setdefault("OMP_WAIT_POLICY", "passive")
        lib = ct.CDLL(_build.build())
        lib.dfjk_oracle_num_threads.restype = ct.c_int
        lib.dfjk_oracle_unpack_slice.argtypes = [ct.c_int, _dp, _dp]
        lib.dfjk_oracle_unpack_slice.restype = None
        lib.dfjk_oracle_density.argtypes = [ct.c_int, ct.c_int, _dp, _dp, _dp]
        lib.dfjk_oracle_density.restype = None
        lib.dfjk_oracle_get_jk.argtypes = [ct.c_int, ct.c_int, ct.c_int, _ip, _dp, _dp, _dp, _dp, _dp, _dp]
        lib.dfjk_oracle_get_jk.restype = ct.c_int
        lib.dfjk_oracle_get_k_dform.argtypes = [ct.c_int, ct.c_int, _dp, _dp, _dp]
        lib.dfjk_oracle_get_k_dform.restype = ct.c_int
        lib.dfjk_oracle_bruteforce.argtypes = [ct.c_int, ct.c_int, _dp, _dp, _dp, _dp]
        lib.dfjk_oracle_bruteforce.restype = ct.c_int
        lib.dfjk_oracle_sample.argtypes = [ct.c_int, ct.c_int, ct.c_int, _ip, _dp, _dp, _dp, ct.c_int,
                                           _ip, _ip, _ip, _dp, _dp]
        lib.dfjk_oracle_sample.restype = ct.c_int
        lib.dfjk_oracle_ao2mo.argtypes = [ct.c_int] * 5 + [_dp] * 6
        lib.dfjk_oracle_ao2mo.restype = ct.c_int
        lib.dfjk_oracle_ao2mo_bruteforce.argtypes = [ct.c_int] * 5 + [_dp] * 4
        lib.dfjk_oracle_ao2mo_bruteforce.restype = ct.c_int
        lib.dfjk_oracle_ao2mo_sample.argtypes = [ct.c_int] * 5 + [_dp, _dp, ct.c_int] + [_ip] * 4 + [_dp, _dp]
        lib.dfjk_oracle_ao2mo_sample.restype = ct.c_int
        _lib = lib
    return _lib


def _d(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(_dp)


def _i(a: np.ndarray):
    return a.ctypes.data_as(_ip)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _concat(Cs: Sequence[np.ndarray], occs: Sequence[np.ndarray], nao: int):
    nocc = np.array([int(np.asarray(o).shape[0]) for o in occs], dtype=np.int32)
    for c, n in zip(Cs, nocc):
        assert np.asarray(c).shape == (nao, n), (np.asarray(c).shape, nao, n)
    C = np.concatenate([_f64(c).ravel() for c in Cs]) if len(Cs) else np.zeros(0)
    occ = np.concatenate([_f64(o).ravel() for o in occs]) if len(occs) else np.zeros(0)
    if C.size == 0:
        C, occ = np.zeros(1), np.zeros(1)
    return nocc, _f64(C), _f64(occ)


def num_threads() -> int:
    return int(_load().dfjk_oracle_num_threads())


def unpack_slice(BpP: np.ndarray, nao: int) -> np.ndarray:
    BpP = _f64(BpP)
    assert BpP.shape == (nao * (nao + 1) // 2,)
    out = np.empty((nao, nao))
    _load().dfjk_oracle_unpack_slice(nao, _d(BpP), _d(out))
    return out


def density(C: np.ndarray, occ: np.ndarray) -> np.ndarray:
    C, occ = _f64(C), _f64(occ)
    nao, nocc = C.shape
    D = np.empty((nao, nao))
    Cq = C if nocc else np.zeros(1)
    oq = occ if nocc else np.zeros(1)
    _load().dfjk_oracle_density(nao, nocc, _d(Cq), _d(oq), _d(D))
    return D


def get_jk(B_packed: np.ndarray, nao: int, Cs: Sequence[np.ndarray], occs: Sequence[np.ndarray],
           with_j: bool = True, with_k: bool = True, with_rho: bool = False):
    """(J, K[, rho]) of every set: J, K are (nset, nao, nao); a skipped output is None."""
    B = _f64(B_packed)
    naux = B.shape[0]
    assert B.ndim == 2 and B.shape[1] == nao * (nao + 1) // 2
    nset = len(Cs)
    nocc, C, occ = _concat(Cs, occs, nao)
    J = np.empty((nset, nao, nao)) if with_j else None
    K = np.empty((nset, nao, nao)) if with_k else None
    rho = np.empty((nset, naux)) if with_rho else None
    Bq = B if B.size else np.zeros(1)
    rc = _load().dfjk_oracle_get_jk(naux, nao, nset, _i(nocc), _d(C), _d(occ), _d(Bq), _d(J), _d(K), _d(rho))
    if rc != 0:
        raise RuntimeError(f"dfjk_oracle_get_jk failed with code {rc}")
    return (J, K, rho) if with_rho else (J, K)


def get_jk_inputs(inp, **kw):
    """get_jk on a dfjk_inputs.DFJKInputs bundle."""
    return get_jk(inp.B_packed, inp.nao, inp.C, inp.occ, **kw)


def get_k_dform(B_packed: np.ndarray, nao: int, D: np.ndarray) -> np.ndarray:
    B, D = _f64(B_packed), _f64(D)
    assert D.shape == (nao, nao)
    K = np.empty((nao, nao))
    rc = _load().dfjk_oracle_get_k_dform(B.shape[0], nao, _d(D), _d(B if B.size else np.zeros(1)), _d(K))
    if rc != 0:
        raise RuntimeError(f"dfjk_oracle_get_k_dform failed with code {rc}")
    return K


def bruteforce(B_packed: np.ndarray, nao: int, D: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    B, D = _f64(B_packed), _f64(D)
    J, K = np.empty((nao, nao)), np.empty((nao, nao))
    rc = _load().dfjk_oracle_bruteforce(B.shape[0], nao, _d(D), _d(B if B.size else np.zeros(1)), _d(J), _d(K))
    if rc != 0:
        raise RuntimeError(f"dfjk_oracle_bruteforce failed with code {rc}")
    return J, K


def sample(B_packed: np.ndarray, nao: int, Cs, occs, samples: Sequence[Tuple[int, int, int]],
           with_j: bool = True, with_k: bool = True):
    """J and K at the listed (set, mu, nu) elements, each from its definition."""
    B = _f64(B_packed)
    nocc, C, occ = _concat(Cs, occs, nao)
    sm = np.ascontiguousarray(np.asarray(samples, dtype=np.int32).reshape(-1, 3))
    ss, mu, nu = (np.ascontiguousarray(sm[:, k]) for k in range(3))
    n = sm.shape[0]
    Jv = np.empty(max(n, 1)) if with_j else None
    Kv = np.empty(max(n, 1)) if with_k else None
    rc = _load().dfjk_oracle_sample(B.shape[0], nao, len(Cs), _i(nocc), _d(C), _d(occ),
                                    _d(B if B.size else np.zeros(1)), n, _i(ss), _i(mu), _i(nu), _d(Jv), _d(Kv))
    if rc != 0:
        raise RuntimeError(f"dfjk_oracle_sample failed with code {rc}")
    return (None if Jv is None else Jv[:n]), (None if Kv is None else Kv[:n])


def ao2mo(B_packed: np.ndarray, nao: int, M: np.ndarray, a0: int, nact: int, with_bmo: bool = False):
    """Eq. 18-21 (oracle/ao2mo_oracle.c): returns (bpa, ppaa, papa[, bmo]) with shapes
    (naux, nmo, nact), (nmo, nmo, nact, nact), (nmo, nact, nmo, nact)[, (naux, nmo, nmo)]."""
    B, M = _f64(B_packed), _f64(M)
    naux, nmo = B.shape[0], M.shape[1]
    assert M.shape[0] == nao and B.shape[1] == nao * (nao + 1) // 2
    bpa = np.empty((naux, nmo, nact))
    ppaa = np.empty((nmo, nmo, nact, nact))
    papa = np.empty((nmo, nact, nmo, nact))
    bmo = np.empty((naux, nmo, nmo)) if with_bmo else None
    z = np.zeros(1)
    rc = _load().dfjk_oracle_ao2mo(naux, nao, nmo, a0, nact, _d(M if M.size else z), _d(B if B.size else z),
                                   _d(bmo), _d(bpa if bpa.size else z), _d(ppaa if ppaa.size else z),
                                   _d(papa if papa.size else z))
    if rc != 0:
        raise RuntimeError(f"dfjk_oracle_ao2mo failed with code {rc}")
    return (bpa, ppaa, papa, bmo) if with_bmo else (bpa, ppaa, papa)


def ao2mo_bruteforce(B_packed: np.ndarray, nao: int, M: np.ndarray, a0: int, nact: int):
    """(ppaa, papa) from the direct 4-index transformation of the Eq. 12 tensor (tiny shapes)."""
    B, M = _f64(B_packed), _f64(M)
    nmo = M.shape[1]
    ppaa = np.empty((nmo, nmo, nact, nact))
    papa = np.empty((nmo, nact, nmo, nact))
    z = np.zeros(1)
    rc = _load().dfjk_oracle_ao2mo_bruteforce(B.shape[0], nao, nmo, a0, nact, _d(M), _d(B if B.size else z),
                                              _d(ppaa if ppaa.size else z), _d(papa if papa.size else z))
    if rc != 0:
        raise RuntimeError(f"dfjk_oracle_ao2mo_bruteforce failed with code {rc}")
    return ppaa, papa


def ao2mo_sample(B_packed: np.ndarray, nao: int, M: np.ndarray, a0: int, nact: int,
                 samples: Sequence[Tuple[int, int, int, int]]):
    """(ppaa[p1][p2][a1][a2], papa[p1][a1][p2][a2]) at the listed (p1, p2, a1, a2), each element from
    the definitions Eq. 18-21 (plain loops over the packed triangle)."""
    B, M = _f64(B_packed), _f64(M)
    nmo = M.shape[1]
    assert M.shape[0] == nao and B.shape[1] == nao * (nao + 1) // 2
    sm = np.ascontiguousarray(np.asarray(samples, dtype=np.int32).reshape(-1, 4))
    cols = [np.ascontiguousarray(sm[:, k]) for k in range(4)]
    n = sm.shape[0]
    v20, v21 = np.empty(max(n, 1)), np.empty(max(n, 1))
    rc = _load().dfjk_oracle_ao2mo_sample(B.shape[0], nao, nmo, a0, nact, _d(M), _d(B if B.size else np.zeros(1)), n,
                                          _i(cols[0]), _i(cols[1]), _i(cols[2]), _i(cols[3]), _d(v20), _d(v21))
    if rc != 0:
        raise RuntimeError(f"dfjk_oracle_ao2mo_sample failed with code {rc}")
    return v20[:n], v21[:n]
