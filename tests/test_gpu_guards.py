"""Guard bands around every buffer the caller hands to the C ABI (compute-sanitizer is not available on the
GPU pool, so the bounds are checked here).

Inputs (B_packed, C, occ, D, M) sit between bands of NaN: a kernel that reads past an end and lets the value
into its arithmetic -- even multiplied by zero -- turns the result into NaN, and a result that depends on what
lies next to an input differs from the run on plain tensors (the calls are deterministic, so the comparison
is bitwise).  Outputs (J, K, bpa, ppaa, papa) sit between bands of a sentinel that must come back untouched.
Covers 16-byte and 8-byte aligned B (an odd offset into the buffer), ragged sizes, the single-launch and the
tiled paths, the density-matrix form, AO2MO and the allocation-free entry point.
"""
import numpy as np
import pytest

import dfjk_inputs

pytestmark = pytest.mark.gpu

BAND = 4096          # doubles on each side
SENTINEL = 12345.678


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device; there is no CPU fallback")
    return torch


def banded(torch, shape, fill, src=None, odd=False):
    """a tensor of `shape` inside a flat buffer with BAND doubles of `fill` on each side (odd: the view starts at
    an odd double, i.e. 8-byte but not 16-byte aligned); returns (view, buffer, offset)"""
    n = int(np.prod(shape)) if len(shape) else 1
    off = BAND + (1 if odd else 0)
    buf = torch.full((off + n + BAND,), fill, dtype=torch.float64, device="cuda")
    view = buf[off:off + n].view(*shape)
    if src is not None:
        view.copy_(src)
    return view, buf, off


def same(torch, a, b, bitwise):
    """bitwise when both runs take the same kernels; an 8-byte aligned B takes other loads (other summation order)"""
    if bitwise:
        return torch.equal(a, b)
    return float((a - b).abs().max()) <= 1e-12 * max(float(b.abs().max()), 1e-300)


def bands_intact(torch, buf, off, n, fill):
    lo, hi = buf[:off], buf[off + n:]
    if fill != fill:
        return bool(torch.isnan(lo).all()) and bool(torch.isnan(hi).all())
    return bool((lo == fill).all()) and bool((hi == fill).all())


CASES = [
    # nao, naux, nocc, odd B offset, handle options
    (48, 33, [12], False, {}),                                   # single launch
    (48, 33, [12], False, {"no_small_path": True}),              # tiled kernels, thin set
    (77, 45, [9, 0, 17], False, {"no_small_path": True}),        # odd npair: 8-byte aligned rows, gathers
    (77, 45, [9, 0, 17], True, {"no_small_path": True}),
    (130, 70, [40, 8], False, {}),                               # even npair: bulk copies, packed pieces (v = 1)
    (130, 70, [40, 8], True, {}),                                # same, B only 8-byte aligned
    (176, 37, [8], False, {}),                                   # one thin set: one-pass half-transform (symm.cu)
    (200, 64, [31, 30, 8], False, {"two_pass_j": True}),         # v = 1, three sets: J pass 1 on the tensor pipe
    (96, 130, [6] * 8, False, {}),                               # eight sets
    (300, 200, [80], False, {}),                                 # small-config shape: packed pieces (v = 3), J pass 1 with 8 rows per CTA
    (360, 150, [100, 8], True, {}),                              # v = 3, 8-byte aligned B
    (424, 96, [200, 9], False, {"nblk": 40}),                    # v = 3, wide N tile, several aux blocks
]


@pytest.mark.parametrize("nao,naux,nocc,odd,opts", CASES)
def test_get_jk_stays_inside_its_buffers(torch_cuda, nao, naux, nocc, odd, opts):
    torch = torch_cuda
    import paper_2505_03755_b200 as pkg
    nan = float("nan")
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed=8800 + nao + naux, L=9.0)
    nset, ntot = len(nocc), sum(nocc)
    B0 = torch.from_numpy(inp.B_packed).cuda()
    C0 = torch.from_numpy(np.concatenate([c.reshape(-1) for c in inp.C])).cuda()
    o0 = torch.from_numpy(np.concatenate(inp.occ)).cuda()
    # reference: plain tensors
    with pkg.DFJK(B0, nao, **opts) as h:
        Jr, Kr = h.get_jk_raw(nocc, C0, o0)
        Jo, _ = h.get_jk_raw(nocc, C0, o0, with_k=False)
        _, Ko = h.get_jk_raw(nocc, C0, o0, with_j=False)
        torch.cuda.synchronize()
    B, Bbuf, Boff = banded(torch, (naux, inp.npair), nan, B0, odd=odd)
    C, Cbuf, Coff = banded(torch, (nao * ntot,), nan, C0)
    occ, obuf, ooff = banded(torch, (ntot,), nan, o0)
    J, Jbuf, Joff = banded(torch, (nset, nao, nao), SENTINEL)
    K, Kbuf, Koff = banded(torch, (nset, nao, nao), SENTINEL)
    with pkg.DFJK(B, nao, **opts) as h:
        for with_j, with_k, Jx, Kx in ((True, True, Jr, Kr), (True, False, Jo, None), (False, True, None, Ko)):
            J.fill_(nan)
            K.fill_(nan)
            h.get_jk_raw(nocc, C, occ, with_j=with_j, with_k=with_k, out_j=J if with_j else None, out_k=K if with_k else None)
            torch.cuda.synchronize()
            if with_j:
                assert bool(torch.isfinite(J).all()) and same(torch, J, Jx, not odd)
            if with_k:
                assert bool(torch.isfinite(K).all()) and same(torch, K, Kx, not odd)
            assert bands_intact(torch, Jbuf, Joff, J.numel(), SENTINEL), "write outside J_out"
            assert bands_intact(torch, Kbuf, Koff, K.numel(), SENTINEL), "write outside K_out"
    for buf, off, n in ((Bbuf, Boff, B.numel()), (Cbuf, Coff, C.numel()), (obuf, ooff, occ.numel())):
        assert bands_intact(torch, buf, off, n, nan), "an input buffer was written"


@pytest.mark.parametrize("nao,naux,odd", [(77, 30, False), (130, 40, True), (64, 20, False)])
def test_get_jk_dm_stays_inside_its_buffers(torch_cuda, nao, naux, odd):
    torch = torch_cuda
    import paper_2505_03755_b200 as pkg
    nan = float("nan")
    inp = dfjk_inputs.make_random(nao, naux, [5], seed=8900 + nao, L=9.0)
    rng = np.random.default_rng(8901 + nao)
    Dn = rng.standard_normal((2, nao, nao))
    Dn = Dn + Dn.transpose(0, 2, 1)
    B0 = torch.from_numpy(inp.B_packed).cuda()
    D0 = torch.from_numpy(Dn).cuda()
    with pkg.DFJK(B0, nao) as h:
        Jr, Kr = h.get_jk_dm(D0)
        torch.cuda.synchronize()
    B, Bbuf, Boff = banded(torch, (naux, inp.npair), nan, B0, odd=odd)
    D, Dbuf, Doff = banded(torch, (2, nao, nao), nan, D0)
    J, Jbuf, Joff = banded(torch, (2, nao, nao), SENTINEL)
    K, Kbuf, Koff = banded(torch, (2, nao, nao), SENTINEL)
    with pkg.DFJK(B, nao) as h:
        h.get_jk_dm(D, out_j=J, out_k=K)
        torch.cuda.synchronize()
    assert bool(torch.isfinite(J).all()) and bool(torch.isfinite(K).all())
    assert same(torch, J, Jr, not odd) and same(torch, K, Kr, not odd)
    assert bands_intact(torch, Jbuf, Joff, J.numel(), SENTINEL) and bands_intact(torch, Kbuf, Koff, K.numel(), SENTINEL)
    assert bands_intact(torch, Bbuf, Boff, B.numel(), nan) and bands_intact(torch, Dbuf, Doff, D.numel(), nan)


@pytest.mark.parametrize("nao,naux,nmo,a0,nact,route", [
    (77, 30, 40, 30, 6, 1), (77, 30, 40, 30, 6, 2), (130, 36, 60, 49, 11, 2), (176, 24, 48, 40, 8, 0),
])
def test_ao2mo_reads_stay_inside_its_inputs(torch_cuda, nao, naux, nmo, a0, nact, route):
    """inputs between NaN bands, outputs compared bitwise with the run on plain tensors"""
    torch = torch_cuda
    import paper_2505_03755_b200 as pkg
    nan = float("nan")
    inp = dfjk_inputs.make_random(nao, naux, [4], seed=9000 + nao + nmo, L=9.0)
    rng = np.random.default_rng(9001 + nao)
    M0 = torch.from_numpy(rng.standard_normal((nao, nmo))).cuda()
    B0 = torch.from_numpy(inp.B_packed).cuda()
    with pkg.DFJK(B0, nao, ao2mo_route=route) as h:
        ref = h.ao2mo(M0, a0, nact)
        torch.cuda.synchronize()
    B, Bbuf, Boff = banded(torch, (naux, inp.npair), nan, B0)
    M, Mbuf, Moff = banded(torch, (nao, nmo), nan, M0)
    with pkg.DFJK(B, nao, ao2mo_route=route) as h:
        out = h.ao2mo(M, a0, nact)
        torch.cuda.synchronize()
    for r, o in zip(ref, out):
        assert bool(torch.isfinite(o).all()) and torch.equal(r, o)
    assert bands_intact(torch, Bbuf, Boff, B.numel(), nan) and bands_intact(torch, Mbuf, Moff, M.numel(), nan)


@pytest.mark.parametrize("nao,naux,nocc,odd", [(48, 33, [12], False), (77, 45, [9, 0, 17], True), (96, 130, [6] * 8, False)])
def test_static_scratch_entry_stays_inside_its_buffers(torch_cuda, nao, naux, nocc, odd):
    torch = torch_cuda
    import paper_2505_03755_b200 as pkg
    nan = float("nan")
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed=9100 + nao, L=9.0)
    nset, ntot = len(nocc), sum(nocc)
    B0 = torch.from_numpy(inp.B_packed).cuda()
    C0 = torch.from_numpy(np.concatenate([c.reshape(-1) for c in inp.C])).cuda()
    o0 = torch.from_numpy(np.concatenate(inp.occ)).cuda()
    Jr = torch.empty((nset, nao, nao), dtype=torch.float64, device="cuda")
    Kr = torch.empty_like(Jr)
    pkg.small_jk_static(B0, nao, nocc, C0, o0, out_j=Jr, out_k=Kr)
    B, Bbuf, Boff = banded(torch, (naux, inp.npair), nan, B0, odd=odd)
    C, Cbuf, Coff = banded(torch, (nao * ntot,), nan, C0)
    occ, obuf, ooff = banded(torch, (ntot,), nan, o0)
    J, Jbuf, Joff = banded(torch, (nset, nao, nao), SENTINEL)
    K, Kbuf, Koff = banded(torch, (nset, nao, nao), SENTINEL)
    pkg.small_jk_static(B, nao, nocc, C, occ, out_j=J, out_k=K)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(J).all()) and bool(torch.isfinite(K).all())
    assert same(torch, J, Jr, not odd) and same(torch, K, Kr, not odd)
    assert bands_intact(torch, Jbuf, Joff, J.numel(), SENTINEL) and bands_intact(torch, Kbuf, Koff, K.numel(), SENTINEL)
    for buf, off, n in ((Bbuf, Boff, B.numel()), (Cbuf, Coff, C.numel()), (obuf, ooff, occ.numel())):
        assert bands_intact(torch, buf, off, n, nan)
