"""ctypes binding of include/dfjk.h (same names, marshalling only).

There is no CPU fallback: if libdfjk.so is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as ct
import os
from typing import List, Optional, Sequence, Tuple

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_NAME = "libdfjk.so"
_lib = None

EXPORTS = ["dfjk_create", "dfjk_get_jk", "dfjk_get_jk_host", "dfjk_destroy", "dfjk_strerror",
           "dfjk_last_error", "dfjk_workspace_bytes", "dfjk_get_plan", "dfjk_last_launch_count",
           "dfjk_selftest_dmma", "dfjk_set_profiling", "dfjk_get_profile", "dfjk_ao2mo", "dfjk_get_jk_dm", "dfjk_last_ao2mo_route",
           "dfjk_small_jk_static", "dfjk_small_jk_static_last_error"]

PHASES = ["prep", "j1", "j2", "j_epilogue", "half_transform", "syrk", "k_epilogue"]


class DFJKError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"dfjk error {code}: {msg}")
        self.code = code


class dfjk_options(ct.Structure):
    _fields_ = [("workspace_cap_bytes", ct.c_size_t), ("nblk", ct.c_int), ("max_nocc_total", ct.c_int),
                ("max_nset", ct.c_int), ("copy_B", ct.c_int), ("ksplit", ct.c_int), ("no_retile", ct.c_int), ("ao2mo_route", ct.c_int), ("two_pass_j", ct.c_int),
                ("k_emulation_slices", ct.c_int), ("k_emulation_group", ct.c_int), ("ht_emulation_slices", ct.c_int),
                ("no_symm_thin", ct.c_int), ("no_small_path", ct.c_int)]


def lib_path() -> str:
    return os.path.join(HERE, _LIB_NAME)


def load_library():
    """Load libdfjk.so (built in-tree by paper_2505_03755_b200.build); fail loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} is missing: run `python -m paper_2505_03755_b200.build` "
                                "(there is no CPU fallback)")
    lib = ct.CDLL(path)
    vp, ip, dp = ct.c_void_p, ct.POINTER(ct.c_int), ct.c_void_p
    lib.dfjk_create.argtypes = [ct.c_int, ct.c_int, dp, ct.POINTER(dfjk_options), ct.POINTER(vp)]
    lib.dfjk_create.restype = ct.c_int
    for name in ("dfjk_get_jk", "dfjk_get_jk_host"):
        fn = getattr(lib, name)
        fn.argtypes = [vp, ct.c_int, ip, dp, dp, dp, dp, vp]
        fn.restype = ct.c_int
    lib.dfjk_get_jk_dm.argtypes = [vp, ct.c_int, dp, dp, dp, vp]
    lib.dfjk_get_jk_dm.restype = ct.c_int
    lib.dfjk_ao2mo.argtypes = [vp, ct.c_int, ct.c_int, ct.c_int, dp, dp, dp, dp, vp]
    lib.dfjk_ao2mo.restype = ct.c_int
    lib.dfjk_destroy.argtypes = [vp]
    lib.dfjk_destroy.restype = ct.c_int
    lib.dfjk_strerror.argtypes = [ct.c_int]
    lib.dfjk_strerror.restype = ct.c_char_p
    lib.dfjk_last_error.argtypes = [vp]
    lib.dfjk_last_error.restype = ct.c_char_p
    lib.dfjk_workspace_bytes.argtypes = [vp]
    lib.dfjk_workspace_bytes.restype = ct.c_size_t
    lib.dfjk_get_plan.argtypes = [vp, ip, ip, ip, ip]
    lib.dfjk_get_plan.restype = ct.c_int
    lib.dfjk_last_launch_count.argtypes = [vp]
    lib.dfjk_last_launch_count.restype = ct.c_int
    lib.dfjk_last_ao2mo_route.argtypes = [vp]
    lib.dfjk_last_ao2mo_route.restype = ct.c_int
    lib.dfjk_set_profiling.argtypes = [vp, ct.c_int]
    lib.dfjk_set_profiling.restype = ct.c_int
    lib.dfjk_get_profile.argtypes = [vp, ct.POINTER(ct.c_double), ip]
    lib.dfjk_get_profile.restype = ct.c_int
    lib.dfjk_selftest_dmma.argtypes = []
    lib.dfjk_selftest_dmma.restype = ct.c_int
    lib.dfjk_small_jk_static.argtypes = [ct.c_int, ct.c_int, dp, ct.c_int, ip, dp, dp, dp, dp, vp]
    lib.dfjk_small_jk_static.restype = ct.c_int
    lib.dfjk_small_jk_static_last_error.argtypes = []
    lib.dfjk_small_jk_static_last_error.restype = ct.c_char_p
    _lib = lib
    return lib


def _check(lib, code: int, handle=None):
    if code != 0:
        msg = lib.dfjk_strerror(code).decode()
        if handle is not None:
            extra = lib.dfjk_last_error(handle).decode()
            if extra:
                msg += f" ({extra})"
        raise DFJKError(code, msg)


def selftest_dmma() -> None:
    lib = load_library()
    _check(lib, lib.dfjk_selftest_dmma())


def small_jk_static(B_packed, nao: int, nocc: List[int], C, occ, out_j=None, out_k=None, stream=None) -> None:
    """dfjk_small_jk_static: the single-launch get_jk on the library's static scratch; no handle and no
    allocation, here or in the library.  C/occ concatenated on the device as for DFJK.get_jk_raw; out_j/out_k
    are caller-allocated (nset, nao, nao) CUDA float64 tensors (None skips that output).  Calls that overlap
    on the GPU race on the shared scratch."""
    import torch
    lib = load_library()
    npair = nao * (nao + 1) // 2
    if not (B_packed.is_cuda and B_packed.dtype == torch.float64 and B_packed.is_contiguous()
            and B_packed.dim() == 2 and B_packed.shape[1] == npair):
        raise ValueError(f"B_packed must be a contiguous CUDA float64 tensor of shape (naux, {npair})")
    nset = len(nocc)
    for t in (out_j, out_k):
        if t is not None and not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                                  and tuple(t.shape) == (nset, nao, nao)):
            raise ValueError(f"outputs must be contiguous CUDA float64 tensors of shape {(nset, nao, nao)}")
    with torch.cuda.device(B_packed.device):
        st = stream if stream is not None else torch.cuda.current_stream()
        arr = (ct.c_int * max(nset, 1))(*nocc)
        code = lib.dfjk_small_jk_static(int(B_packed.shape[0]), int(nao), ct.c_void_p(B_packed.data_ptr()), nset, arr,
                                        ct.c_void_p(C.data_ptr()), ct.c_void_p(occ.data_ptr()),
                                        ct.c_void_p(out_j.data_ptr() if out_j is not None else 0),
                                        ct.c_void_p(out_k.data_ptr() if out_k is not None else 0),
                                        ct.c_void_p(st.cuda_stream))
    if code != 0:
        msg = lib.dfjk_strerror(code).decode()
        extra = lib.dfjk_small_jk_static_last_error().decode()
        raise DFJKError(code, f"{msg} ({extra})" if extra else msg)


class DFJK:
    """Handle on a resident packed tensor B (torch CUDA float64, shape (naux, nao(nao+1)/2))."""

    def __init__(self, B_packed, nao: int, *, workspace_cap_bytes: int = 0, nblk: int = 0,
                 max_nocc_total: int = 0, max_nset: int = 0, copy_B: bool = False, ksplit: int = 0,
                 two_pass_j: bool = False, no_retile: bool = False, ao2mo_route: int = 0,
                 k_emulation_slices: int = 0, k_emulation_group: int = 0, ht_emulation_slices: int = 0,
                 no_symm_thin: bool = False, no_small_path: bool = False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("dfjk needs a CUDA device (sm_100); there is no CPU fallback")
        self._lib = load_library()
        if not (B_packed.is_cuda and B_packed.dtype == torch.float64 and B_packed.is_contiguous()):
            raise ValueError("B_packed must be a contiguous CUDA float64 tensor")
        npair = nao * (nao + 1) // 2
        if B_packed.dim() != 2 or B_packed.shape[1] != npair:
            raise ValueError(f"B_packed must have shape (naux, {npair})")
        self.naux, self.nao, self.npair = int(B_packed.shape[0]), int(nao), npair
        self._B = None if copy_B else B_packed      # borrowed: keep it alive
        self._device = B_packed.device
        opt = dfjk_options(workspace_cap_bytes, nblk, max_nocc_total, max_nset, int(copy_B), ksplit, int(no_retile), int(ao2mo_route), int(two_pass_j),
                           int(k_emulation_slices), int(k_emulation_group), int(ht_emulation_slices), int(no_symm_thin), int(no_small_path))
        h = ct.c_void_p()
        with torch.cuda.device(self._device):
            code = self._lib.dfjk_create(self.naux, self.nao, ct.c_void_p(B_packed.data_ptr() if self.naux else 0),
                                         ct.byref(opt), ct.byref(h))
        _check(self._lib, code)
        self._h = h

    # -- marshalling helpers
    @staticmethod
    def _concat(Cs, occs, nao, device, torch):
        nocc = [int(o.shape[0]) for o in occs]
        for c, n in zip(Cs, nocc):
            if tuple(c.shape) != (nao, n):
                raise ValueError(f"C block has shape {tuple(c.shape)}, expected {(nao, n)}")
        if sum(nocc) == 0:
            z = torch.zeros(1, dtype=torch.float64, device=device)
            return nocc, z, z
        C = torch.cat([c.to(device=device, dtype=torch.float64).contiguous().reshape(-1) for c in Cs])
        occ = torch.cat([o.to(device=device, dtype=torch.float64).reshape(-1) for o in occs])
        return nocc, C, occ

    def get_jk(self, Cs: Sequence, occs: Sequence, with_j: bool = True, with_k: bool = True,
               out_j=None, out_k=None, stream=None):
        """J, K (nset, nao, nao) of D_s = C_s diag(occ_s) C_s^T; enqueue-only on `stream`."""
        import torch
        with torch.cuda.device(self._device):
            st = stream if stream is not None else torch.cuda.current_stream()
            # the concatenated temporaries are produced, consumed and released on `st`
            with torch.cuda.stream(st):
                nocc, C, occ = self._concat(Cs, occs, self.nao, self._device, torch)
                return self.get_jk_raw(nocc, C, occ, with_j, with_k, out_j, out_k, st)

    def get_jk_raw(self, nocc: List[int], C, occ, with_j=True, with_k=True, out_j=None, out_k=None, stream=None):
        """Same, with C/occ already concatenated on the device (no torch ops in the call path)."""
        import torch
        nset = len(nocc)
        with torch.cuda.device(self._device):
            st = stream if stream is not None else torch.cuda.current_stream()
            J = out_j if out_j is not None else (torch.empty((nset, self.nao, self.nao), dtype=torch.float64, device=self._device) if with_j else None)
            K = out_k if out_k is not None else (torch.empty((nset, self.nao, self.nao), dtype=torch.float64, device=self._device) if with_k else None)
            arr = (ct.c_int * max(nset, 1))(*nocc)
            code = self._lib.dfjk_get_jk(self._h, nset, arr, ct.c_void_p(C.data_ptr()), ct.c_void_p(occ.data_ptr()),
                                         ct.c_void_p(J.data_ptr() if J is not None else 0),
                                         ct.c_void_p(K.data_ptr() if K is not None else 0),
                                         ct.c_void_p(st.cuda_stream))
        _check(self._lib, code, self._h)
        return J, K

    def get_jk_host(self, nocc: List[int], C_host, occ_host, J_host=None, K_host=None, stream=None):
        """dfjk_get_jk_host: C/occ/J/K are HOST (ideally pinned) float64 tensors; synchronises."""
        import torch
        nset = len(nocc)
        with torch.cuda.device(self._device):
            st = stream if stream is not None else torch.cuda.current_stream()
            arr = (ct.c_int * max(nset, 1))(*nocc)
            code = self._lib.dfjk_get_jk_host(self._h, nset, arr, ct.c_void_p(C_host.data_ptr()),
                                              ct.c_void_p(occ_host.data_ptr()),
                                              ct.c_void_p(J_host.data_ptr() if J_host is not None else 0),
                                              ct.c_void_p(K_host.data_ptr() if K_host is not None else 0),
                                              ct.c_void_p(st.cuda_stream))
        _check(self._lib, code, self._h)
        return J_host, K_host

    def get_jk_dm(self, D, with_j: bool = True, with_k: bool = True, out_j=None, out_k=None, stream=None):
        """dfjk_get_jk_dm: D is a CUDA float64 (nset, nao, nao) tensor of symmetric density matrices
        (Eq. 14-17 as printed); returns (J, K), enqueue-only."""
        import torch
        if D.dim() != 3 or tuple(D.shape[1:]) != (self.nao, self.nao):
            raise ValueError(f"D must have shape (nset, {self.nao}, {self.nao})")
        nset = int(D.shape[0])
        with torch.cuda.device(self._device):
            st = stream if stream is not None else torch.cuda.current_stream()
            with torch.cuda.stream(st):            # a converted copy of D lives and dies on `st`
                D = D.to(device=self._device, dtype=torch.float64).contiguous()
                J = out_j if out_j is not None else (torch.empty_like(D) if with_j else None)
                K = out_k if out_k is not None else (torch.empty_like(D) if with_k else None)
                code = self._lib.dfjk_get_jk_dm(self._h, nset, ct.c_void_p(D.data_ptr()),
                                                ct.c_void_p(J.data_ptr() if J is not None else 0),
                                                ct.c_void_p(K.data_ptr() if K is not None else 0),
                                                ct.c_void_p(st.cuda_stream))
        _check(self._lib, code, self._h)
        return J, K

    def ao2mo(self, M, a0: int, nact: int, with_ppaa: bool = True, with_papa: bool = True, stream=None):
        """dfjk_ao2mo (Eq. 18-21): M is a CUDA float64 (nao, nmo) tensor; returns (bpa, ppaa, papa) with
        shapes (naux, nmo, nact), (nmo, nmo, nact, nact), (nmo, nact, nmo, nact); enqueue-only."""
        import torch
        if tuple(M.shape[:1]) != (self.nao,) or M.dim() != 2:
            raise ValueError(f"M must have shape ({self.nao}, nmo)")
        nmo = int(M.shape[1])
        with torch.cuda.device(self._device):
            st = stream if stream is not None else torch.cuda.current_stream()
            with torch.cuda.stream(st):            # a converted copy of M lives and dies on `st`
                M = M.to(device=self._device, dtype=torch.float64).contiguous()
                kw = dict(dtype=torch.float64, device=self._device)
                bpa = torch.empty((self.naux, nmo, nact), **kw)
                ppaa = torch.empty((nmo, nmo, nact, nact), **kw) if with_ppaa else None
                papa = torch.empty((nmo, nact, nmo, nact), **kw) if with_papa else None
                code = self._lib.dfjk_ao2mo(self._h, nmo, a0, nact, ct.c_void_p(M.data_ptr() if nmo else 0),
                                            ct.c_void_p(bpa.data_ptr() if bpa.numel() else 0),
                                            ct.c_void_p(ppaa.data_ptr() if ppaa is not None and ppaa.numel() else 0),
                                            ct.c_void_p(papa.data_ptr() if papa is not None and papa.numel() else 0),
                                            ct.c_void_p(st.cuda_stream))
        _check(self._lib, code, self._h)
        return bpa, ppaa, papa

    def plan(self) -> dict:
        a, b, c, d = ct.c_int(), ct.c_int(), ct.c_int(), ct.c_int()
        _check(self._lib, self._lib.dfjk_get_plan(self._h, ct.byref(a), ct.byref(b), ct.byref(c), ct.byref(d)))
        return dict(nblk=a.value, ksplit=b.value, nocc_pad_capacity=c.value, retiled=d.value)

    def set_profiling(self, on: bool) -> None:
        _check(self._lib, self._lib.dfjk_set_profiling(self._h, int(on)), self._h)

    def profile(self) -> dict:
        """{phase: (ms, launch groups)} of the last get_jk (synchronises on its last event)."""
        ms = (ct.c_double * len(PHASES))()
        n = (ct.c_int * len(PHASES))()
        _check(self._lib, self._lib.dfjk_get_profile(self._h, ms, n), self._h)
        return {p: (ms[i], n[i]) for i, p in enumerate(PHASES)}

    @property
    def workspace_bytes(self) -> int:
        return int(self._lib.dfjk_workspace_bytes(self._h))

    @property
    def last_ao2mo_route(self) -> int:
        return int(self._lib.dfjk_last_ao2mo_route(self._h))

    @property
    def last_launch_count(self) -> int:
        return int(self._lib.dfjk_last_launch_count(self._h))

    def close(self):
        if getattr(self, "_h", None):
            self._lib.dfjk_destroy(self._h)
            self._h = None
            self._B = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


def get_jk(B_packed, nao: int, Cs, occs, **kw) -> Tuple:
    """One-shot convenience: create, get_jk, destroy."""
    import torch
    with DFJK(B_packed, nao) as h:
        J, K = h.get_jk(Cs, occs, **kw)
        torch.cuda.current_stream().synchronize()
    return J, K
